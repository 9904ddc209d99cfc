"""Seeded synthetic inputs for the TQP routed-expert layer (serves BOTH the oracle and the CUDA path).

This module holds none of the method's arithmetic: it only draws random tensors in the storage
formats the layer's boundary uses (bf16 / fp16 bit patterns, uint8 codes, fp32 router weights) and
names the five BASELINE.json configs (plus one extra measurement shape).  Recipe: SURVEY.md §8(d) / DESIGN.md "Input recipe".

bf16 tensors are carried as numpy uint16 bit patterns (numpy has no bf16); fp16 as numpy float16.
"""
from __future__ import annotations

import dataclasses

import numpy as np


@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    T: int
    d: int
    F: int
    E: int
    k: int
    r: int
    seed: int
    skew: bool = False          # cfg 3: additive Zipf(1.1) logit bias over a seeded permutation
    backward: bool = True
    router_grad: bool = False   # cfg 0 / cfg 4: dtopk_w, dW_r and the router term of dX
    lora_scale: float = 1.0

    @property
    def N(self) -> int:
        return self.T * self.k


CONFIGS = {
    0: Config("cfg0_tiny", T=64, d=128, F=256, E=8, k=2, r=8, seed=0, router_grad=True),
    1: Config("cfg1_9b", T=4096, d=2048, F=1024, E=64, k=8, r=16, seed=1, backward=False),
    2: Config("cfg2_120b", T=8192, d=2560, F=1024, E=460, k=12, r=16, seed=2),
    3: Config("cfg3_120b_skew", T=8192, d=2560, F=1024, E=460, k=12, r=16, seed=3, skew=True),
    4: Config("cfg4_120b_mb", T=16384, d=2560, F=1024, E=460, k=12, r=32, seed=4, router_grad=True),
    # extra measurement shape (not a BASELINE.json config): the paper's own 120B layer width, d_model = 4096
    # (Table 33)
    5: Config("cfg5_120b_d4096", T=8192, d=4096, F=1024, E=460, k=12, r=16, seed=5),
}


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16, returned as uint16 bit patterns (finite inputs)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    rounding = ((u >> 16) & 1) + np.uint32(0x7FFF)
    return ((u + rounding) >> 16).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    """Exact widening bf16 bit patterns -> fp32."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32)


def _normal_bf16(rng: np.random.Generator, shape, std: float) -> np.ndarray:
    return f32_to_bf16_bits(rng.standard_normal(shape, dtype=np.float32) * np.float32(std))


def zipf_logit_bias(E: int, seed: int, s: float = 1.1) -> np.ndarray:
    """cfg 3: bias[pi(i)] = log p_i, p_i ∝ i^-s, pi a seeded permutation of the experts."""
    rng = np.random.default_rng(10_000 + seed)
    ranks = np.arange(1, E + 1, dtype=np.float64)
    p = ranks ** (-s)
    p /= p.sum()
    pi = rng.permutation(E)
    bias = np.empty(E, dtype=np.float32)
    bias[pi] = np.log(p).astype(np.float32)
    return bias


def make_inputs(cfg: Config, *, T: int | None = None, E: int | None = None) -> dict:
    """Draw every tensor of one layer call.  `T`/`E` override the config (bounded samples)."""
    T = cfg.T if T is None else T
    E = cfg.E if E is None else E
    d, F, r = cfg.d, cfg.F, cfg.r
    rng = np.random.default_rng(cfg.seed)
    out = {
        "T": T, "d": d, "F": F, "E": E, "k": cfg.k, "r": r, "lora_scale": float(cfg.lora_scale),
        "X": _normal_bf16(rng, (T, d), 1.0),                                   # bf16 bits [T,d]
        "dY": _normal_bf16(rng, (T, d), 1.0),                                  # bf16 bits [T,d]
        "W_r": (rng.standard_normal((d, E), dtype=np.float32) * np.float32(0.02)),  # fp32 [d,E]
        "codebook": (rng.standard_normal((256, 8), dtype=np.float32) * np.float32(0.02)).astype(np.float16),
        "idx_gate": rng.integers(0, 256, size=(E, F, d // 8), dtype=np.uint8),
        "idx_up": rng.integers(0, 256, size=(E, F, d // 8), dtype=np.uint8),
        "idx_down": rng.integers(0, 256, size=(E, d, F // 8), dtype=np.uint8),
        "scale_gate": rng.uniform(0.5, 1.5, size=(E, F)).astype(np.float16),
        "scale_up": rng.uniform(0.5, 1.5, size=(E, F)).astype(np.float16),
        "scale_down": rng.uniform(0.5, 1.5, size=(E, d)).astype(np.float16),
        "A_gate": _normal_bf16(rng, (E, d, r), 0.01),
        "B_gate": _normal_bf16(rng, (E, r, F), 0.01),
        "A_up": _normal_bf16(rng, (E, d, r), 0.01),
        "B_up": _normal_bf16(rng, (E, r, F), 0.01),
        "A_down": _normal_bf16(rng, (E, F, r), 0.01),
        "B_down": _normal_bf16(rng, (E, r, d), 0.01),
        "logit_bias": zipf_logit_bias(E, cfg.seed) if cfg.skew else None,
    }
    return out
