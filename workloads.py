"""Seeded synthetic input generators for the five StreamKL workloads (BASELINE.json `configs`).

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA path
(`paper_2606_20005_b200/`).  It holds none of the method's arithmetic: it draws random
numbers, rounds them once to the storage dtype and hands out raw arrays.

Recipe (stands in for the paper's own synthetic sweep):
  per (cfg, b, h) an independent stream  PCG64(SeedSequence([2606_20005, cfg, b, h])),
  draw order  Q1f, K1f, Q2f|eps_q, K2f|eps_k, g  -- float32 standard normals (g is U(0.5,1.5)),
  then one rounding to the config dtype (bf16 round-to-nearest-even, or kept fp32).

bf16 tensors are carried as uint16 bit patterns (numpy has no bf16); `bf16_to_f32` widens exactly.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace

import numpy as np

ROOT_SEED = 2606_20005


@dataclass(frozen=True)
class Config:
    """One workload. `near` = cfg-2 recipe (Q2=Q1+0.1*eps), `q1_scale` = cfg-5 peaky logits."""

    idx: int
    name: str
    B: int
    H: int
    NQ: int
    NK: int
    d1: int
    d2: int
    dtype: str  # "bf16" | "f16" | "f32"
    causal: bool
    near: bool = False
    q1_scale: float = 1.0
    teacher_grads: bool = True  # does the backward also produce dQ1,dK1?
    unit_dkl: bool = False  # cfg 1 is specified with dkl_rows = 1

    @property
    def c1(self) -> float:
        return 1.0 / math.sqrt(self.d1)

    @property
    def c2(self) -> float:
        return 1.0 / math.sqrt(self.d2)

    @property
    def BH(self) -> int:
        return self.B * self.H

    def visible_pairs(self) -> int:
        """Number of (query,key) pairs inside the mask, exact (bottom-right aligned causal)."""
        if not self.causal:
            return self.BH * self.NQ * self.NK
        off = self.NK - self.NQ  # row i sees keys 0..i+off  (i+off+1 <= NK for every row)
        return self.BH * (self.NQ * (off + 1) + self.NQ * (self.NQ - 1) // 2)

    def visible_pairs_convention(self) -> float:
        """(query,key) pairs under BASELINE.json's FLOP convention: NQ*NK per head, halved for causal."""
        p = float(self.BH) * self.NQ * self.NK
        return p / 2 if self.causal else p

    def fwd_flop(self) -> float:
        """BASELINE.json convention: 2*NQ*NK*(d1+d2) per head, halved for causal."""
        f = 2.0 * self.BH * self.NQ * self.NK * (self.d1 + self.d2)
        return f / 2 if self.causal else f

    def bwd_flop(self) -> float:
        """One-visit GEMM count: recompute (d1+d2) + 2*d2 (dQ2,dK2) [+ 2*d1 (dQ1,dK1)] MAC per pair."""
        mac = (self.d1 + self.d2) + 2 * self.d2 + (2 * self.d1 if self.teacher_grads else 0)
        f = 2.0 * self.BH * self.NQ * self.NK * mac
        return f / 2 if self.causal else f


CONFIGS = {
    1: Config(1, "tiny", 1, 1, 256, 256, 64, 64, "f32", False, teacher_grads=False, unit_dkl=True),
    2: Config(2, "near-identical", 1, 32, 4096, 4096, 128, 128, "bf16", True, near=True),
    3: Config(3, "indexer", 1, 32, 16384, 16384, 128, 64, "bf16", True, teacher_grads=False),
    4: Config(4, "long-context", 1, 32, 65536, 65536, 128, 128, "bf16", True),
    5: Config(5, "skewed", 4, 16, 2048, 131072, 128, 64, "bf16", False, q1_scale=4.0),
}


def shrink(cfg: Config, **kw) -> Config:
    """Same recipe at another size (parity cases the oracle finishes in seconds)."""
    return replace(cfg, **kw)


# --------------------------------------------------------------------------------------
# bf16 <-> f32 bit handling (storage only)
# --------------------------------------------------------------------------------------
def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16, returned as uint16 bit patterns."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    lsb = (u >> np.uint32(16)) & np.uint32(1)
    r = u + np.uint32(0x7FFF) + lsb
    return (r >> np.uint32(16)).astype(np.uint16)


def bf16_to_f32(bits: np.ndarray) -> np.ndarray:
    return (bits.astype(np.uint32) << np.uint32(16)).view(np.float32)


def widen_f64(a: np.ndarray) -> np.ndarray:
    """Exact widening of a stored tensor (uint16 bf16 bits, float16 or float32) to float64."""
    if a.dtype == np.uint16:
        return bf16_to_f32(a).astype(np.float64)
    return a.astype(np.float64)


def _store(x: np.ndarray, dtype: str) -> np.ndarray:
    if dtype == "bf16":
        return f32_to_bf16_bits(x)
    if dtype == "f32":
        return np.ascontiguousarray(x, dtype=np.float32)
    if dtype == "f16":
        return np.ascontiguousarray(x, dtype=np.float32).astype(np.float16)   # IEEE round-to-nearest-even
    raise ValueError(dtype)


# --------------------------------------------------------------------------------------
# generation
# --------------------------------------------------------------------------------------
def head_inputs(cfg: Config, b: int, h: int):
    """Inputs of ONE (b,h): dict Q1 [NQ,d1], K1 [NK,d1], Q2 [NQ,d2], K2 [NK,d2] (stored dtype), g [NQ] f32."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([ROOT_SEED, cfg.idx, b, h])))
    f32 = np.float32
    Q1f = rng.standard_normal((cfg.NQ, cfg.d1), dtype=f32)
    K1f = rng.standard_normal((cfg.NK, cfg.d1), dtype=f32)
    if cfg.q1_scale != 1.0:
        Q1f *= f32(cfg.q1_scale)
    if cfg.near:
        if cfg.d1 != cfg.d2:
            raise ValueError("near-identical recipe needs d1 == d2")
        Q2f = Q1f + f32(0.1) * rng.standard_normal((cfg.NQ, cfg.d2), dtype=f32)
        K2f = K1f + f32(0.1) * rng.standard_normal((cfg.NK, cfg.d2), dtype=f32)
    else:
        Q2f = rng.standard_normal((cfg.NQ, cfg.d2), dtype=f32)
        K2f = rng.standard_normal((cfg.NK, cfg.d2), dtype=f32)
    if cfg.unit_dkl:
        g = np.ones(cfg.NQ, dtype=f32)
    else:
        g = (f32(0.5) + rng.random(cfg.NQ, dtype=f32)).astype(f32)
    return {
        "Q1": _store(Q1f, cfg.dtype),
        "K1": _store(K1f, cfg.dtype),
        "Q2": _store(Q2f, cfg.dtype),
        "K2": _store(K2f, cfg.dtype),
        "g": g,
    }


def all_inputs(cfg: Config, heads=None):
    """Stack heads into [B,H,N,d] arrays (or [len(heads),N,d] when an explicit (b,h) list is given)."""
    if heads is None:
        heads = [(b, h) for b in range(cfg.B) for h in range(cfg.H)]
        shape = (cfg.B, cfg.H)
    else:
        shape = (len(heads),)
    st = {"bf16": np.uint16, "f16": np.float16, "f32": np.float32}[cfg.dtype]
    out = {
        "Q1": np.empty(shape + (cfg.NQ, cfg.d1), st),
        "K1": np.empty(shape + (cfg.NK, cfg.d1), st),
        "Q2": np.empty(shape + (cfg.NQ, cfg.d2), st),
        "K2": np.empty(shape + (cfg.NK, cfg.d2), st),
        "g": np.empty(shape + (cfg.NQ,), np.float32),
    }
    for n, (b, h) in enumerate(heads):
        one = head_inputs(cfg, b, h)
        ix = np.unravel_index(n, shape)
        for k, v in one.items():
            out[k][ix] = v
    return out
