"""Pins for the LSE merge (merging partials equals attention over the full range;
the reduction is associative)."""
import math

import numpy as np

import oracle

RNG = np.random.default_rng(7)


def rand16(*shape):
    return RNG.standard_normal(shape).astype(np.float16)


def test_hand_example():
    # (lse, o) = (ln 3, 2) (+) (ln 1, 10) = (ln 4, 4)
    o, lse = oracle.merge(np.array([[[2.0]], [[10.0]]]), np.array([[math.log(3)], [0.0]]))
    assert abs(lse[0] - math.log(4)) < 1e-15 and abs(o[0, 0] - 4.0) < 1e-14


def test_single_partial_is_identity():
    op = RNG.standard_normal((1, 5, 128))
    lp = RNG.standard_normal((1, 5))
    o, lse = oracle.merge(op, lp)
    assert np.array_equal(o, op[0]) and np.array_equal(lse, lp[0])


def test_weights_sum_to_one_and_minus_inf():
    lp = np.array([[0.3], [-np.inf], [2.0], [-5.0]])
    op = np.array([[[1.0]], [[np.nan]], [[1.0]], [[1.0]]])  # garbage o for the empty partial
    o, lse = oracle.merge(op, lp)
    assert abs(o[0, 0] - 1.0) < 1e-15  # constant o -> weights sum to 1, NaN ignored
    assert abs(lse[0] - math.log(math.exp(0.3) + math.exp(2.0) + math.exp(-5.0))) < 1e-14
    o2, lse2 = oracle.merge(np.zeros((2, 1, 4)), np.full((2, 1), -np.inf))
    assert lse2[0] == -np.inf and np.array_equal(o2, np.zeros((1, 4)))


def _split_attend(q, K, V, cuts):
    edges = [0] + list(cuts) + [K.shape[1]]
    ops, lps = [], []
    for a, b in zip(edges[:-1], edges[1:]):
        o, l = oracle.attend(q, K, V, t_begin=a, t_end=b)
        ops.append(o)
        lps.append(l)
    return np.stack(ops), np.stack(lps)


def test_any_split_equals_unsplit():
    Hq, Hkv, S = 8, 2, 500
    q, K, V = rand16(Hq, 128), rand16(Hkv, S, 128), rand16(Hkv, S, 128)
    o_full, lse_full = oracle.attend(q, K, V)
    for nparts in (1, 2, 3, 7, 32):
        cuts = sorted(RNG.choice(np.arange(1, S), size=nparts - 1, replace=False).tolist())
        op, lp = _split_attend(q, K, V, cuts)
        o, lse = oracle.merge(op, lp)
        assert np.abs(o - o_full).max() < 1e-12 and np.abs(lse - lse_full).max() < 1e-12
    # 1-token parts at both ends
    op, lp = _split_attend(q, K, V, [1, 2, S - 1])
    o, lse = oracle.merge(op, lp)
    assert np.abs(o - o_full).max() < 1e-12 and np.abs(lse - lse_full).max() < 1e-12


def test_merge_order_and_tree_shape():
    Hq, S = 4, 256
    q, K, V = rand16(Hq, 128), rand16(1, S, 128), rand16(1, S, 128)
    op, lp = _split_attend(q, K, V, [10, 50, 51, 130, 200])
    o_flat, l_flat = oracle.merge(op, lp)
    perm = RNG.permutation(op.shape[0])
    o_p, l_p = oracle.merge(op[perm], lp[perm])
    assert np.abs(o_p - o_flat).max() < 1e-13 and np.abs(l_p - l_flat).max() < 1e-13
    # binary tree: ((0,1),(2,3)),(4,5)
    def m2(a, b):
        o, l = oracle.merge(np.stack([a[0], b[0]]), np.stack([a[1], b[1]]))
        return o, l
    leaves = [(op[i], lp[i]) for i in range(6)]
    t = m2(m2(m2(leaves[0], leaves[1]), m2(leaves[2], leaves[3])), m2(leaves[4], leaves[5]))
    assert np.abs(t[0] - o_flat).max() < 1e-13 and np.abs(t[1] - l_flat).max() < 1e-13
    # left fold
    acc = leaves[0]
    for x in leaves[1:]:
        acc = m2(acc, x)
    assert np.abs(acc[0] - o_flat).max() < 1e-13 and np.abs(acc[1] - l_flat).max() < 1e-13


def test_triple_form_conversion():
    # PAPER.md:145 partials are (o_i, m_i, l_i); any m_i >= max is a valid triple and
    # l_i * exp(m_i) = exp(lse_i) (reading 3)
    q, K, V = rand16(1, 128), rand16(1, 64, 128), rand16(1, 64, 128)
    o, lse = oracle.attend(q, K, V)
    s = (K[0].astype(np.float64) @ q[0].astype(np.float64)) / math.sqrt(128)
    for m in (s.max(), s.max() + 3.0):
        l = np.exp(s - m).sum()
        assert abs(math.log(l) + m - lse[0]) < 1e-13
