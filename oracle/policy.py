"""Algorithm 1 of the paper ("A-node scaling policy"), step by step -- TEST INFRASTRUCTURE.

Plain Python floats (fp64), written in the paper's order and notation so that it can be checked against the text by
eye.  Shares nothing with the library's controller (csrc/kf_policy.cu).

Readings (rows 20-22):
  * "2B" in C_total is two bytes per fp16 element, not the batch size.
  * g_i of line 11 is the q_i of line 8: the growth of node i in bytes per step (the listing is garbled, :199-:204);
    H_kn in Eq. 2 is H_kv (:238).
  * "no pending prewarm for i" (l.12): a prewarm that is already READY but not yet published also blocks a new one.
  * KVBytes(A_i) counts committed tokens resident on node i times the per-token bytes of all L layers.
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import List, Sequence, Tuple


@dataclass
class PolicyConstants:
    beta_mem: float
    beta_slo: float
    gamma: float
    t_a_max_s: float      # T_A^max, seconds
    bw_hbm: float         # BW_HBM, bytes / s
    c_kv_cap: float       # C_kv_cap, bytes
    t_step_s: float       # T_step
    t_prewarm_s: float    # T_prewarm
    n_kv_heads: int       # H_kv
    head_dim: int         # d_h
    n_layers: int         # L


def bytes_per_token(c: PolicyConstants) -> float:
    """2 * H_kv * d_h * L * 2B."""
    return 2 * c.n_kv_heads * c.head_dim * c.n_layers * 2


def threshold(c: PolicyConstants) -> float:
    """Line 1 / Eq. (1): C_thresh = min(beta_mem * C_kv_cap, beta_slo * T_A^max * BW_HBM)."""
    return min(c.beta_mem * c.c_kv_cap, c.beta_slo * c.t_a_max_s * c.bw_hbm)


def initial_nodes(c: PolicyConstants, s: Sequence[int]) -> int:
    """Lines 2-3: C_total = sum_i 2 s_i H_kv d_h L * 2B ;  N_A = ceil(C_total / C_thresh)."""
    c_total = sum(s_i * bytes_per_token(c) for s_i in s)
    return math.ceil(c_total / threshold(c))


def monitor(c: PolicyConstants, tokens: Sequence[int], tails: Sequence[int], prewarm_pending: Sequence[bool],
            prewarm_ready: Sequence[bool]) -> List[Tuple[float, bool, bool]]:
    """Lines 6-19, one pass.  Returns per node (tau_fill, spawn a prewarm, publish the route at the next boundary)."""
    c_thresh = threshold(c)
    out = []
    for i in range(len(tokens)):
        tau, spawn, publish = math.inf, False, False
        if tails[i] > 0:                                            # l.6  foreach tail-holding A-node i
            n_i = tails[i]                                          # l.7
            q_i = n_i * bytes_per_token(c)                          # l.8  growth per step (= g_i)
            b_i = tokens[i] * bytes_per_token(c)                    # l.9  KVBytes(A_i)
            if q_i > 0:                                             # l.10
                tau = (c_thresh - b_i) / q_i                        # l.11 Eq. (2)
                if tau * c.t_step_s < c.t_prewarm_s and not prewarm_pending[i] and not prewarm_ready[i]:
                    spawn = True                                    # l.12-13
            if b_i >= c.gamma * c_thresh and prewarm_ready[i]:      # l.16
                publish = True                                      # l.17
        out.append((tau, spawn, publish))
    return out
