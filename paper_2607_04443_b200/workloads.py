"""Seeded synthetic inputs with the shapes of BASELINE.json's five configs.

This module is the ONE thing the CUDA path's tests/bench and the CPU oracle's tests share.
It holds none of the method's arithmetic (no attention, no relayout, no cache write): only
shapes, seeds, value distributions and BF16 input rounding.  It imports neither the CUDA
binding nor oracle/.

Recipe: rng = numpy.random.default_rng(seed);
float32 standard_normal draws in this fixed order -- Q, K_cache prefill, V_cache prefill,
K_slice, V_slice, K_new, V_new, then (multi-step configs) Q, K_new, V_new for steps 1.. --
then scaling (q_premul, kv_std), then round-to-nearest-even to BF16 where dtype == "bf16".
The paper fixes only the resolutions and the 160 ms unit; every size here
is BASELINE.json's "illustrative" one.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional, Tuple

import numpy as np


@dataclasses.dataclass(frozen=True)
class UnitConfig:
    name: str
    seed: int
    dtype: str  # "bf16" | "f32"
    H: int  # heads the attention call handles (after any seq->head relayout)
    d: int
    q_block_end: Tuple[int, ...]  # block-causal mask: block b covers query rows [q_block_end[b-1], q_block_end[b])
    kv_visible: Tuple[int, ...]  # ... and sees keys j < kv_visible[b] on the timeline cache ++ new
    cache_prefill: int  # rows already in the cache before this unit's write
    capacity: int
    write_rows: int = 0  # K/V slice rows written at write_offset before attention
    write_offset: int = 0
    Ln: int = 0  # rows of the unit's own K/V passed next to the cache
    softmax_scale: float = 1.0
    q_premul: float = 1.0  # Q is multiplied by this BEFORE rounding (config 2)
    kv_std: float = 1.0
    steps: int = 1  # denoising steps per unit (config 5: 8), each with its own Q/K_new/V_new
    # Ulysses-rank emulation (config 4): Q/K_new/V_new are drawn as [L, H_full, d] and relaid
    P: int = 1
    g0: int = 0
    G: int = 1
    H_full: Optional[int] = None
    note: str = ""

    @property
    def Lq(self) -> int:
        return self.q_block_end[-1]

    @property
    def cache_len(self) -> int:
        """Valid cache rows when attention runs (after the write)."""
        return max(self.cache_prefill, self.write_offset + self.write_rows) if self.write_rows else self.cache_prefill

    @property
    def elem_bytes(self) -> int:
        return 2 if self.dtype == "bf16" else 4

    def visible_pairs(self) -> int:
        """Pi = sum_b |block b| * kv_visible[b]  (per head)."""
        prev, tot = 0, 0
        for e, v in zip(self.q_block_end, self.kv_visible):
            tot += (e - prev) * v
            prev = e
        return tot

    def attn_flops(self) -> int:
        """Algorithmic flops of ONE attention call: 4 * Pi * d * H (visible pairs only)."""
        return 4 * self.visible_pairs() * self.d * self.H


def _cfg4(name, seed, L_unit, units, H_full, P, g0, d, cache, note):
    L = L_unit * units
    return UnitConfig(name=name, seed=seed, dtype="bf16", H=H_full // P, d=d,
                      q_block_end=tuple(L_unit * (u + 1) for u in range(units)),
                      kv_visible=tuple(cache + L_unit * (u + 1) for u in range(units)),
                      cache_prefill=cache, capacity=cache, Ln=L, softmax_scale=1.0 / math.sqrt(d),
                      P=P, g0=g0, G=1, H_full=H_full, note=note)


CONFIGS = {
    # -- BASELINE.json configs[0]: literal reading (own rows written into the cache, then Ln = 0)
    "cfg1": UnitConfig("cfg1", 0, "f32", H=2, d=64, q_block_end=(32, 64), kv_visible=(160, 192), cache_prefill=128,
                       capacity=256, write_rows=64, write_offset=128, Ln=0, softmax_scale=1.0 / 8.0,
                       note="tiny oracle check; R2 literal reading"),
    # -- same problem with the unit's own K/V passed separately (R2 equivalent reading)
    "cfg1_split": UnitConfig("cfg1_split", 0, "f32", H=2, d=64, q_block_end=(32, 64), kv_visible=(160, 192),
                             cache_prefill=128, capacity=256, Ln=64, softmax_scale=1.0 / 8.0,
                             note="tiny oracle check; own K/V separate"),
    "cfg2": UnitConfig("cfg2", 1, "bf16", H=24, d=128, q_block_end=(292,), kv_visible=(8192 + 292,), cache_prefill=8192,
                       capacity=8192, Ln=292, softmax_scale=1.0, q_premul=1.0 / math.sqrt(128.0),
                       note="v0.1-shaped 192x336 unit: 252 video + 40 audio queries"),
    "cfg3": UnitConfig("cfg3", 2, "bf16", H=40, d=128, q_block_end=(970,), kv_visible=(16384 + 970,), cache_prefill=15360,
                       capacity=16384, write_rows=1024, write_offset=15360, Ln=970, softmax_scale=1.0 / math.sqrt(128.0),
                       note="640x368 unit: 920 video + 50 audio queries; the headline workload"),
    "cfg4": _cfg4("cfg4", 3, 920, 4, 40, 4, 1, 128, 16384, "single Ulysses-rank emulation, P=4"),
    "cfg5": UnitConfig("cfg5", 4, "bf16", H=40, d=128, q_block_end=(970,), kv_visible=(65536 + 970,), cache_prefill=64566,
                       capacity=65536, write_rows=970, write_offset=64566, Ln=970, softmax_scale=1.0 / math.sqrt(128.0),
                       kv_std=0.5, steps=8, note="long-context stress: 8 denoising steps under one CUDA graph"),
    # ---- reduced copies the oracle finishes in seconds; same structure, several tiles + ragged tails ----
    "cfg2_small": UnitConfig("cfg2_small", 1, "bf16", H=3, d=128, q_block_end=(292,), kv_visible=(1000 + 292,),
                             cache_prefill=1000, capacity=1024, Ln=292, softmax_scale=1.0,
                             q_premul=1.0 / math.sqrt(128.0)),
    "cfg3_small": UnitConfig("cfg3_small", 2, "bf16", H=4, d=128, q_block_end=(970,), kv_visible=(2048 + 970,),
                             cache_prefill=1536, capacity=2048, write_rows=512, write_offset=1536, Ln=970,
                             softmax_scale=1.0 / math.sqrt(128.0)),
    "cfg4_small": _cfg4("cfg4_small", 3, 230, 4, 8, 4, 1, 128, 1200, "P=4 emulation, reduced"),
    "cfg5_small": UnitConfig("cfg5_small", 4, "bf16", H=4, d=128, q_block_end=(970,), kv_visible=(4096 + 970,),
                             cache_prefill=3126, capacity=4096, write_rows=970, write_offset=3126, Ln=970,
                             softmax_scale=1.0 / math.sqrt(128.0), kv_std=0.5, steps=3),
}


def bf16_round(x: np.ndarray) -> np.ndarray:
    """Round float32 to the nearest BF16 (ties to even); result is float32 holding exact BF16 values."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    bits = x.view(np.uint32)
    bias = np.uint32(0x7FFF) + ((bits >> np.uint32(16)) & np.uint32(1))
    out = ((bits + bias) & np.uint32(0xFFFF0000)).astype(np.uint32)
    return out.view(np.float32)


def bf16_bits(x: np.ndarray) -> np.ndarray:
    """uint16 bit patterns of float32 values that are already exact BF16."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    return (x.view(np.uint32) >> np.uint32(16)).astype(np.uint16)


def bf16_from_bits(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def device_array(x: np.ndarray, dtype: str) -> np.ndarray:
    """The byte image the GPU receives: uint16 BF16 bits, or float32."""
    return bf16_bits(x) if dtype == "bf16" else np.ascontiguousarray(x, dtype=np.float32)


def generate(cfg: UnitConfig) -> dict:
    """All inputs of one unit as float32 arrays holding exactly the values the GPU receives.

    Keys: q[s], k_new[s], v_new[s] (lists over steps; [L, H_full or H, d]), k_cache, v_cache
    ([H, capacity, d]; rows >= cache_prefill are zero), k_slice, v_slice ([write_rows, H, d] or None).
    """
    rng = np.random.default_rng(cfg.seed)
    Hq = cfg.H_full if cfg.H_full is not None else cfg.H
    L = cfg.Lq

    def draw(shape, scale=1.0):
        x = rng.standard_normal(shape, dtype=np.float32)
        if scale != 1.0:
            x = x * np.float32(scale)
        return bf16_round(x) if cfg.dtype == "bf16" else x

    out = {"q": [], "k_new": [], "v_new": []}
    out["q"].append(draw((L, Hq, cfg.d), cfg.q_premul))
    k_cache = np.zeros((cfg.H, cfg.capacity, cfg.d), np.float32)
    v_cache = np.zeros((cfg.H, cfg.capacity, cfg.d), np.float32)
    k_cache[:, :cfg.cache_prefill] = draw((cfg.H, cfg.cache_prefill, cfg.d), cfg.kv_std)
    v_cache[:, :cfg.cache_prefill] = draw((cfg.H, cfg.cache_prefill, cfg.d), cfg.kv_std)
    out["k_cache"], out["v_cache"] = k_cache, v_cache
    if cfg.write_rows:
        out["k_slice"] = draw((cfg.write_rows, cfg.H, cfg.d), cfg.kv_std)
        out["v_slice"] = draw((cfg.write_rows, cfg.H, cfg.d), cfg.kv_std)
    else:
        out["k_slice"] = out["v_slice"] = None
    if cfg.Ln:
        out["k_new"].append(draw((cfg.Ln, Hq, cfg.d), cfg.kv_std))
        out["v_new"].append(draw((cfg.Ln, Hq, cfg.d), cfg.kv_std))
    for _ in range(1, cfg.steps):
        out["q"].append(draw((L, Hq, cfg.d), cfg.q_premul))
        if cfg.Ln:
            out["k_new"].append(draw((cfg.Ln, Hq, cfg.d), cfg.kv_std))
            out["v_new"].append(draw((cfg.Ln, Hq, cfg.d), cfg.kv_std))
    return out


def sample_pairs(cfg: UnitConfig, n: int, seed: int = 12345):
    """n distinct-ish (row, head) pairs for sampled full-size parity; always includes the first and
    last row of every block and the rows either side of each 128-row tile edge near them."""
    rng = np.random.default_rng(seed + cfg.seed)
    rows = list(rng.integers(0, cfg.Lq, size=n))
    heads = list(rng.integers(0, cfg.H, size=n))
    prev = 0
    for e in cfg.q_block_end:
        for r in (prev, e - 1, min(prev + 127, e - 1), min(prev + 128, e - 1)):
            rows.append(r)
            heads.append(int(rng.integers(0, cfg.H)))
        prev = e
    return np.asarray(rows, np.int32), np.asarray(heads, np.int32)
