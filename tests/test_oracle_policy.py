"""Pins of oracle/policy.py (Algorithm 1) against what the paper and arithmetic fix, and the
library's host-side controller (kf_policy_*) against the oracle.  No GPU needed."""
import math
import random

import pytest

from oracle.policy import PolicyConstants, bytes_per_token, initial_nodes, monitor, threshold

GiB = 1 << 30


def consts(**kw):
    base = dict(beta_mem=1.0, beta_slo=1.0, gamma=0.9, t_a_max_s=1.0, bw_hbm=1e30, c_kv_cap=4096 * 1000.0,
                t_step_s=0.05, t_prewarm_s=0.412, n_kv_heads=8, head_dim=128, n_layers=1)
    base.update(kw)
    return PolicyConstants(**base)


def test_bytes_per_token_llama_8b():
    # 2 * s * H_kv * d_h * L * 2B; Llama-3.1-8B: H_kv = 8, d_h = 128, L = 32 -> 128 KiB per token,
    # and the paper's own sanity figure (:35): batch 64 x 4K tokens = 32 GiB
    c = consts(n_layers=32)
    assert bytes_per_token(c) == 128 * 1024
    assert 64 * 4096 * bytes_per_token(c) == 32 * GiB
    assert bytes_per_token(consts(n_layers=1)) == 4096          # per layer: the 4096 B/token of the hot path


def test_eq1_takes_the_tighter_bound():
    # memory-bound: 0.9 * 40 GB = 36 GB < 0.8 * 0.1 s * 768 GB/s = 61.44 GB
    assert threshold(consts(beta_mem=0.9, c_kv_cap=40e9, beta_slo=0.8, t_a_max_s=0.1, bw_hbm=768e9)) == 0.9 * 40e9
    # SLO-bound: 0.8 * 2 ms * 768 GB/s = 1.2288 GB < 36 GB
    assert threshold(consts(beta_mem=0.9, c_kv_cap=40e9, beta_slo=0.8, t_a_max_s=2e-3, bw_hbm=768e9)) == \
        pytest.approx(1.2288e9, rel=1e-12)
    # T = C / BW_HBM: scanning C_slo at BW_HBM takes beta_slo * T_A^max
    c = consts(beta_slo=0.8, t_a_max_s=2e-3, bw_hbm=768e9, c_kv_cap=1e30)
    assert threshold(c) / c.bw_hbm == pytest.approx(0.8 * 2e-3, rel=1e-12)


def test_initial_nodes_is_a_ceiling():
    c = consts(n_layers=32, c_kv_cap=48.0 * GiB)               # C_thresh = 48 GiB, 128 KiB per token
    per_node = 48 * GiB // (128 * 1024)                        # tokens that fit one node
    assert initial_nodes(c, [per_node * 7]) == 7               # exact multiple: no extra node
    assert initial_nodes(c, [per_node * 7, 1]) == 8            # one token more: one node more
    assert initial_nodes(c, [1]) == 1 and initial_nodes(c, []) == 0
    assert initial_nodes(c, [per_node] * 3 + [per_node // 2] * 2) == 4


def test_eq2_fill_horizon_hand_example():
    # C_thresh = 1000 tokens' worth; node 0 holds 400 tokens and 3 tails -> (1000 - 400) / 3 = 200 steps;
    # node 1 holds tokens but no tail: not monitored
    c = consts()
    out = monitor(c, [400, 900], [3, 0], [False, False], [False, False])
    assert out[0] == (200.0, False, False)
    assert out[1] == (math.inf, False, False)


def test_fill_horizon_drops_by_one_per_step():
    c = consts()
    taus = [monitor(c, [100 + 4 * t], [4], [False], [False])[0][0] for t in range(10)]   # 4 tails: +4 tokens / step
    assert all(taus[t] - taus[t + 1] == 1.0 for t in range(9))


def test_prewarm_trigger_and_blockers():
    # T_prewarm = 412 ms (cold bring-up), T_step = 50 ms -> spawn once tau_fill < 8.24 steps
    c = consts()
    at = lambda tok, pend=False, ready=False: monitor(c, [tok], [1], [pend], [ready])[0]
    assert at(1000 - 9)[1] is False and at(1000 - 9)[0] == 9.0
    assert at(1000 - 8)[1] is True
    assert at(1000 - 8, pend=True)[1] is False                # a pending prewarm blocks a second one
    assert at(1000 - 8, ready=True)[1] is False               # so does a ready, unpublished one (reading)
    assert at(1005)[0] == -5.0 and at(1005)[1] is True        # already over budget: negative horizon, still spawns


def test_publish_needs_watermark_and_ready_prewarm():
    c = consts(gamma=0.9)                                      # watermark at 900 tokens' worth
    at = lambda tok, ready, tails=1: monitor(c, [tok], [tails], [False], [ready])[0][2]
    assert at(899, True) is False
    assert at(900, True) is True                               # >= : equality publishes
    assert at(950, False) is False                             # not ready: wait
    assert at(950, True, tails=0) is False                     # no tail on the node: nothing to redirect


# ---- the library's controller (host code of libkflume) against the oracle ------------------------------------------
def _lib_policy(c):
    from paper_2606_29207_b200 import Policy
    return Policy(beta_mem=c.beta_mem, beta_slo=c.beta_slo, gamma=c.gamma, t_a_max_s=c.t_a_max_s, bw_hbm=c.bw_hbm,
                  c_kv_cap=c.c_kv_cap, t_step_s=c.t_step_s, t_prewarm_s=c.t_prewarm_s, n_kv_heads=c.n_kv_heads,
                  head_dim=c.head_dim, n_layers=c.n_layers)


def test_library_controller_equals_oracle():
    rnd = random.Random(11)
    for _ in range(200):
        c = consts(beta_mem=rnd.uniform(0.5, 1), beta_slo=rnd.uniform(0.5, 1), gamma=rnd.uniform(0.5, 1),
                   t_a_max_s=rnd.uniform(1e-4, 1e-2), bw_hbm=rnd.uniform(5e11, 8e12), c_kv_cap=rnd.uniform(1e9, 2e11),
                   t_step_s=rnd.uniform(0.01, 0.1), t_prewarm_s=rnd.uniform(0.0, 1.0),
                   n_kv_heads=rnd.choice([8, 32, 48]), n_layers=rnd.choice([1, 32, 80]))
        pol = _lib_policy(c)
        assert pol.bytes_per_token() == bytes_per_token(c)
        assert pol.threshold() == threshold(c)
        lens = [rnd.randrange(0, 300000) for _ in range(rnd.randrange(0, 40))]
        assert pol.initial_nodes(lens) == initial_nodes(c, lens)
        P = rnd.randrange(1, 17)
        cap_tok = int(threshold(c) / bytes_per_token(c))
        tokens = [rnd.randrange(0, max(2, int(1.2 * cap_tok))) for _ in range(P)]
        tails = [rnd.choice([0, 0, 1, 3, 17]) for _ in range(P)]
        pend = [rnd.random() < 0.3 for _ in range(P)]
        ready = [rnd.random() < 0.3 for _ in range(P)]
        assert pol.step(tokens, tails, pend, ready) == monitor(c, tokens, tails, pend, ready)


def test_library_controller_rejects_bad_constants():
    from paper_2606_29207_b200 import KFlumeError
    pol = _lib_policy(consts(gamma=0.0))
    assert pol.threshold() == 0.0 and pol.initial_nodes([5]) == -1
    with pytest.raises(KFlumeError):
        pol.step([1], [1], [0], [0])
