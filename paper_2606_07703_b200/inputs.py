"""Seeded synthetic inputs for the five BASELINE.json configs (and small test variants).

This module is the ONE thing the CUDA path's tests/bench and the CPU oracle's tests share.  It holds
none of the method's arithmetic: it only draws numbers (numpy Philox), plants the salience structure
the configs describe, rounds fp32 -> bf16 once (round-to-nearest-even) and returns the bit patterns
as uint16 numpy arrays.  The identical bytes go to the oracle and to the device.

The inputs are synthetic stand-ins for the paper's workloads (Qwen-family GQA layers on RULER-style
long-context prompts), whose prompts, checkpoints and indexer weights are
not available; shapes follow the paper's regime (head dim 128, GQA 4:1, the k schedule PAPER.md:176,
b_sel = 64 PAPER.md:178, d_idx in {128, 64} PAPER.md:280).  The recipe is stated in DESIGN.md.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Dict, Optional, Tuple

import numpy as np

SEED_BASE = 26060770300
T_X, T_WQI, T_WKI, T_Q, T_K, T_V, T_U, T_SAL = range(8)
_CHUNK = 1 << 22  # elements per draw; fixed so the stream does not depend on the caller


@dataclass(frozen=True)
class Config:
    """Problem statement of one layer call + input recipe."""
    name: str
    cfg_id: int
    mode: str                 # "oracle" | "indexer"
    L: int
    Hq: int
    Hkv: int
    d: int
    k: int
    b_sel: int = 1
    hidden: int = 0
    d_idx: int = 0
    salience: bool = False
    local_window: int = 0
    local_bias: float = 0.0
    cu_seqlens: Optional[Tuple[int, ...]] = None
    seed_extra: int = 0
    flags: int = 0            # served-scorer switches: 1 ReLU, 2 key LayerNorm, 4 RoPE

    @property
    def scale(self) -> float:
        return 1.0 / math.sqrt(self.d)

    @property
    def idx_scale(self) -> float:
        return 1.0 / math.sqrt(self.d_idx) if self.d_idx else 0.0

    @property
    def seq_bounds(self):
        cu = self.cu_seqlens if self.cu_seqlens is not None else (0, self.L)
        return [(cu[i], cu[i + 1]) for i in range(len(cu) - 1)]

    @property
    def num_rows(self) -> int:
        b = max(1, self.b_sel)
        return sum((e - s + b - 1) // b for s, e in self.seq_bounds)

    def seed(self, tensor_id: int) -> int:
        return SEED_BASE + 100 * self.cfg_id + tensor_id + self.seed_extra


# BASELINE.json configs, in order.  c4 is a sweep (one Config per length); c5 has a varlen companion.
C1 = Config("c1", 1, "oracle", L=1024, Hq=8, Hkv=2, d=64, k=256, b_sel=1)
C2 = Config("c2", 2, "indexer", L=8192, Hq=16, Hkv=4, d=128, k=1024, b_sel=64, hidden=1024, d_idx=64,
            salience=True)
C3 = Config("c3", 3, "indexer", L=32768, Hq=32, Hkv=8, d=128, k=2048, b_sel=64, hidden=4096, d_idx=128,
            salience=True, local_window=128, local_bias=1.0)
C4_SWEEP = tuple(
    Config(f"c4_{L}", 4, "both", L=L, Hq=32, Hkv=8, d=128, k=k, b_sel=1, hidden=4096, d_idx=128,
           salience=True, seed_extra=L)
    for L, k in ((4096, 256), (8192, 512), (16384, 1024), (32768, 2048), (65536, 2048)))
C5 = Config("c5", 5, "indexer", L=131072, Hq=32, Hkv=8, d=128, k=2048, b_sel=128, hidden=4096, d_idx=128,
            salience=True, local_window=128, local_bias=1.0)
C5_VARLEN = Config("c5_varlen", 5, "indexer", L=40960, Hq=32, Hkv=8, d=128, k=2048, b_sel=128, hidden=4096,
                   d_idx=128, salience=True, local_window=128, local_bias=1.0,
                   cu_seqlens=(0, 16384, 28672, 36864, 40960), seed_extra=50)

ALL = {c.name: c for c in (C1, C2, C3, *C4_SWEEP, C5, C5_VARLEN)}


def shrink(cfg: Config, L: int, **kw) -> Config:
    """A smaller problem with the same recipe (for tests the oracle can finish in seconds)."""
    return replace(cfg, name=f"{cfg.name}_L{L}", L=L, seed_extra=cfg.seed_extra + 7 * L, **kw)


def f32_to_bf16(x: np.ndarray) -> np.ndarray:
    """fp32 -> bf16 bit patterns, round-to-nearest-even (no NaN inputs here)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = (u + (np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1)))) >> np.uint32(16)
    return r.astype(np.uint16)


def bf16_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def _normal(seed: int, shape, sigma: float = 1.0) -> np.ndarray:
    """N(0, sigma^2) fp32 draws from Philox(seed), in fixed-size chunks."""
    rng = np.random.Generator(np.random.Philox(seed))
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.float32)
    for i in range(0, n, _CHUNK):
        j = min(n, i + _CHUNK)
        rng.standard_normal(j - i, dtype=np.float32, out=out[i:j])
    if sigma != 1.0:
        out *= np.float32(sigma)
    return out.reshape(shape)


def _normal_bf16(seed: int, shape, sigma: float = 1.0) -> np.ndarray:
    """Same stream as _normal, converted chunk-wise to bf16 (keeps the fp32 copy out of memory)."""
    rng = np.random.Generator(np.random.Philox(seed))
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.uint16)
    buf = np.empty(min(n, _CHUNK), dtype=np.float32)
    for i in range(0, n, _CHUNK):
        j = min(n, i + _CHUNK)
        b = buf[: j - i]
        rng.standard_normal(j - i, dtype=np.float32, out=b)
        if sigma != 1.0:
            b *= np.float32(sigma)
        out[i:j] = f32_to_bf16(b)
    return out.reshape(shape)


def salient_positions(cfg: Config) -> np.ndarray:
    """round(0.01 * n) distinct positions per sequence, by a seeded permutation (packed positions)."""
    rng = np.random.Generator(np.random.Philox(cfg.seed(T_SAL)))
    out = []
    for s, e in cfg.seq_bounds:
        n = e - s
        m = int(round(0.01 * n))
        out.append(np.sort(rng.permutation(n)[:m]) + s)
    return np.concatenate(out).astype(np.int64) if out else np.empty(0, np.int64)


def make_inputs(cfg: Config, with_indexer: Optional[bool] = None) -> Dict[str, np.ndarray]:
    """Q [L,Hq,d], K,V [L,Hkv,d] (+ X [L,hidden], Wqi, Wki [hidden,d_idx]) as bf16 bit patterns (uint16)."""
    if with_indexer is None:
        with_indexer = cfg.mode in ("indexer", "both") and cfg.hidden > 0
    q = _normal(cfg.seed(T_Q), (cfg.L, cfg.Hq, cfg.d))
    k = _normal(cfg.seed(T_K), (cfg.L, cfg.Hkv, cfg.d))
    out: Dict[str, np.ndarray] = {}
    if cfg.salience:
        u = _normal(cfg.seed(T_U), (cfg.d,)).astype(np.float64)
        u = (u / np.linalg.norm(u)).astype(np.float32)
        q += u                                  # every Q head row += u
        sal = salient_positions(cfg)
        k[sal] += np.float32(3.0) * u           # every KV head's K row at a salient position += 3u
        out["u"] = u
        out["salient"] = sal
    out["Q"] = f32_to_bf16(q)
    del q
    out["K"] = f32_to_bf16(k)
    del k
    out["V"] = _normal_bf16(cfg.seed(T_V), (cfg.L, cfg.Hkv, cfg.d))
    if with_indexer:
        sig = 1.0 / math.sqrt(cfg.hidden)       # N(0, 1/hidden): the second argument is the variance
        out["X"] = _normal_bf16(cfg.seed(T_X), (cfg.L, cfg.hidden))
        out["Wqi"] = _normal_bf16(cfg.seed(T_WQI), (cfg.hidden, cfg.d_idx), sig)
        out["Wki"] = _normal_bf16(cfg.seed(T_WKI), (cfg.hidden, cfg.d_idx), sig)
    return out
