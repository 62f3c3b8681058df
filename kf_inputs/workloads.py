"""Synthetic workload recipes for the five BASELINE.json configs.

Only shapes and per-request context lengths live here -- no arithmetic of the method.  These seeded
synthetic inputs STAND IN FOR the paper's Codex/SWE-bench-Pro serving trace (median
~80K tokens, tails >200K: PAPER.md:33,:349) and for Llama-3.1-8B/70B activations;
neither the trace nor the weights are in this container and neither is reconstructed.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List

import numpy as np

from . import gen

K = 1024


@dataclass
class Workload:
    name: str
    n_q_heads: int
    n_kv_heads: int
    range_tokens: int          # R
    n_partitions: int          # P
    contexts: List[int]        # S_r: tokens resident AT ATTEND TIME of decode step 0 (current token included)
    n_layers: int = 1          # logical layers
    n_steps: int = 1
    head_dim: int = 128
    note: str = ""
    seed: int = gen.SEED
    extra: dict = field(default_factory=dict)

    @property
    def batch(self) -> int:
        return len(self.contexts)

    @property
    def group(self) -> int:
        return self.n_q_heads // self.n_kv_heads

    def max_ranges(self, steps: int | None = None) -> int:
        steps = self.n_steps if steps is None else steps
        return max(1, max(-(-(s + steps - 1) // self.range_tokens) for s in self.contexts))

    def total_ranges(self, steps: int | None = None) -> int:
        steps = self.n_steps if steps is None else steps
        return sum(-(-(s + steps - 1) // self.range_tokens) for s in self.contexts)

    def slots_per_partition(self, steps: int | None = None) -> int:
        # global round-robin => partition p gets ceil or floor of total/P ranges
        return -(-self.total_ranges(steps) // self.n_partitions)

    def kv_bytes_per_token(self) -> int:
        """Per-layer KV bytes per context token = 2 * H_kv * d * 2 B."""
        return 2 * self.n_kv_heads * self.head_dim * 2


def cfg3_lengths(batch: int = 16, seed: int = gen.SEED) -> List[int]:
    """Log-normal contexts, median 80K = 81920, sigma 0.55, clipped to [1K, 200K]."""
    key = gen.stream_key(seed, gen.STREAM_LEN_CFG3)
    h = gen.hash64(key, np.arange(batch, dtype=np.uint64))
    c = 1.0 / math.sqrt(8 * (256 ** 2 - 1) / 12.0)
    # the fp32 constant of normal16 is used so host and any other implementation agree bit for bit
    c32 = float(np.array([0x3B9CC4BF], dtype=np.uint32).view(np.float32)[0])
    assert abs(c - c32) < 1e-9
    out = []
    for s in gen.byte_sum(h):
        z = float(np.float32(np.float32(int(s) - 1020) * np.float32(c32)))
        S = int(round(81920.0 * math.exp(0.55 * z)))
        out.append(min(max(S, 1 * K), 200 * K))
    return out


def cfg5_lengths(batch: int = 128, range_tokens: int = 16 * K, lo: int = 1 * K, hi: int = 128 * K,
                 seed: int = gen.SEED, crosser_every: int = 8, crosser_step: int = 4,
                 max_full_ranges: int = 7) -> List[int]:
    """Uniform [lo, hi] contexts BEFORE step 0, with forced boundary crossers:
    every request with r % 8 == 0 gets length (min(S//R, 7)+1)*R - 4*(r/8), so that exactly one new
    range opens at step 4*(r/8)."""
    key = gen.stream_key(seed, gen.STREAM_LEN_CFG5)
    h = gen.hash64(key, np.arange(batch, dtype=np.uint64))
    span = np.uint64(hi - lo + 1)
    lens = [int(lo + int(x % span)) for x in h]
    R = range_tokens
    for r in range(0, batch, crosser_every):
        k = crosser_step * (r // crosser_every)
        lens[r] = (min(lens[r] // R, max_full_ranges) + 1) * R - k
    return lens


def cfg1() -> Workload:
    return Workload("cfg1", 32, 8, 2 * K, 2, [4096],
                    note="B=1, Llama-3.1-8B shape, context 4096 = 2 ranges of 2048 on 2 partitions")


def cfg2() -> Workload:
    return Workload("cfg2", 32, 8, 4 * K, 1, [4096] * 64,
                    note="B=64, 8B shape, uniform 4096 context, 1 partition, 4096-token ranges")


def cfg3() -> Workload:
    return Workload("cfg3", 32, 8, 32 * K, 8, cfg3_lengths(),
                    note="B=16, 8B shape, log-normal contexts (median 80K, clip 200K), 32K ranges, 8 partitions")


def cfg4() -> Workload:
    return Workload("cfg4", 64, 8, 32 * K, 32, [K * K],
                    note="B=1, Llama-3.1-70B shape (G=8), context 1,048,576 = 32 ranges of 32K on 32 partitions")


def cfg5() -> Workload:
    # contexts here are S_r(0)+1: cfg5_lengths() is the context BEFORE step 0
    lens = cfg5_lengths()
    return Workload("cfg5", 32, 8, 16 * K, 16, [s + 1 for s in lens], n_layers=32, n_steps=64,
                    note="B=128, 8B shape, contexts U[1K,128K] + 16 forced range-fill events, 16K ranges, "
                         "16 partitions, 64 steps x 32 layers",
                    extra={"len_before_step0": lens})


def cfg5_twin() -> Workload:
    """1/16-scale parity twin of cfg5 with truly distinct layers."""
    lens = cfg5_lengths(batch=128, range_tokens=1 * K, lo=64, hi=8 * K)
    return Workload("cfg5_twin", 32, 8, 1 * K, 16, [s + 1 for s in lens], n_layers=32, n_steps=64,
                    note="cfg5 at 1/16 scale: contexts U[64,8K], R=1K, same forced-event rule, 32 distinct layers",
                    extra={"len_before_step0": lens})


def tiny_t0() -> Workload:
    """SURVEY Appendix B tiny case T0: H_q=8, H_kv=2, S=5, R=4."""
    return Workload("t0", 8, 2, 4, 2, [5], note="tiny: ranges [0,4) and [4,5)")


FIG10_HEADS = [(32, 8), (48, 8), (64, 8), (32, 32), (40, 40), (48, 48)]   # PAPER.md:322 (Fig. 10)


def fig10(n_q_heads: int, n_kv_heads: int, batch: int, seq: int, range_tokens: int = 8 * K,
          n_partitions: int = 4) -> Workload:
    """Head-shape sweep of the paper's Fig. 10: six head configurations (GQA Q32:KV8, Q48:KV8,
    Q64:KV8; MHA Q32:KV32, Q40:KV40, Q48:KV48), batch 8-128, sequence 2K-32K; every request at context `seq`, KV cut
    into 8K-token ranges routed round-robin over 4 emulated attention nodes."""
    assert (n_q_heads, n_kv_heads) in FIG10_HEADS and 8 <= batch <= 128 and 2 * K <= seq <= 32 * K
    return Workload(f"fig10_q{n_q_heads}kv{n_kv_heads}_b{batch}_s{seq // K}k", n_q_heads, n_kv_heads, range_tokens,
                    n_partitions, [seq] * batch,
                    note=f"Fig. 10 shape Q{n_q_heads}:KV{n_kv_heads}, batch {batch}, every request at context {seq}, "
                         f"{range_tokens // K}K ranges over {n_partitions} partitions")


def by_name(name: str) -> Workload:
    if name.startswith("fig10_"):      # fig10_q<Hq>kv<Hkv>_b<batch>_s<seq in K>k
        import re
        m = re.fullmatch(r"fig10_q(\d+)kv(\d+)_b(\d+)_s(\d+)k", name)
        if not m:
            raise KeyError(name)
        return fig10(int(m.group(1)), int(m.group(2)), int(m.group(3)), int(m.group(4)) * K)
    return {"cfg1": cfg1, "cfg2": cfg2, "cfg3": cfg3, "cfg4": cfg4, "cfg5": cfg5,
            "cfg5_twin": cfg5_twin, "t0": tiny_t0}[name]()
