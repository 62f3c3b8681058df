"""Pins for oracle/attention.c: closed forms, invariants, library routines, brute force, golden values.

Each test is chosen so that a plausible mistake in the oracle (dropped scale, wrong sign, transposed
operand, wrong head mapping, un-normalised output, log base) fails at least one of them."""
import math

import numpy as np
import pytest

import oracle
from kf_inputs import gen
from conftest import load_golden

RNG = np.random.default_rng(20260629)


def rand16(*shape, scale=1.0):
    return (RNG.standard_normal(shape) * scale).astype(np.float16)


# ---------------------------------------------------------------- closed forms ------------------
def test_one_token_context_returns_v():
    q, K, V = rand16(8, 128), rand16(2, 1, 128), rand16(2, 1, 128)
    o, lse = oracle.attend(q, K, V)
    for h in range(8):
        assert np.array_equal(o[h], V[h // 4, 0].astype(np.float64))
        s = (q[h].astype(np.float64) @ K[h // 4, 0].astype(np.float64)) / math.sqrt(128)
        assert abs(lse[h] - s) < 1e-13


def test_identical_keys_return_mean_v():
    S = 37
    q = rand16(4, 128)
    k0 = rand16(1, 1, 128)
    K = np.repeat(k0, S, axis=1)
    V = rand16(1, S, 128)
    o, lse = oracle.attend(q, K, V)
    mean = V[0].astype(np.float64).mean(axis=0)
    for h in range(4):
        assert np.abs(o[h] - mean).max() < 1e-14
        s = (q[h].astype(np.float64) @ k0[0, 0].astype(np.float64)) / math.sqrt(128)
        assert abs(lse[h] - (s + math.log(S))) < 1e-13


def test_zero_query():
    S = 100
    q = np.zeros((4, 128), np.float16)
    K, V = rand16(2, S, 128), rand16(2, S, 128)
    o, lse = oracle.attend(q, K, V)
    assert np.allclose(lse, math.log(S), atol=1e-14)
    for h in range(4):
        assert np.abs(o[h] - V[h // 2].astype(np.float64).mean(axis=0)).max() < 1e-14


def test_two_tokens_sigmoid():
    q, K, V = rand16(2, 128), rand16(1, 2, 128), rand16(1, 2, 128)
    o, lse = oracle.attend(q, K, V, scale=0.25)
    for h in range(2):
        s = 0.25 * (K[0].astype(np.float64) @ q[h].astype(np.float64))
        w1 = 1.0 / (1.0 + math.exp(-(s[1] - s[0])))
        expect = (1 - w1) * V[0, 0].astype(np.float64) + w1 * V[0, 1].astype(np.float64)
        assert np.abs(o[h] - expect).max() < 1e-14
        assert abs(lse[h] - (s[0] + math.log1p(math.exp(s[1] - s[0])))) < 1e-13


def test_hand_example_d1():
    # SURVEY 8(c) pin (v): d=1, scale=1, q=[1], K=[0, ln2, ln3], V=[6,12,18] -> weights 1/6,2/6,3/6
    # (fp16 rounding of ln2/ln3 is accounted for by computing the expectation from the rounded keys)
    q = np.array([[1.0]], np.float16)
    K = np.array([[[0.0], [math.log(2)], [math.log(3)]]], np.float16)
    V = np.array([[[6.0], [12.0], [18.0]]], np.float16)
    o, lse = oracle.attend(q, K, V, scale=1.0)
    e = np.exp(K[0, :, 0].astype(np.float64))
    assert abs(lse[0] - math.log(e.sum())) < 1e-14
    assert abs(o[0, 0] - (e * np.array([6.0, 12.0, 18.0])).sum() / e.sum()) < 1e-13
    # and against the exact textbook numbers, within the fp16 rounding of ln2, ln3 (<= 2^-11 relative)
    assert abs(lse[0] - math.log(6)) < 1e-3
    assert abs(o[0, 0] - 14.0) < 1e-2


def test_hand_example_exact_powers_of_two():
    # exactly representable: scores ln-free.  q=[1], K=[0,1,2] scale=ln2 -> weights 1,2,4 /7
    q = np.array([[1.0]], np.float16)
    K = np.array([[[0.0], [1.0], [2.0]]], np.float16)
    V = np.array([[[7.0], [14.0], [-7.0]]], np.float16)
    o, lse = oracle.attend(q, K, V, scale=math.log(2))
    assert abs(lse[0] - math.log(7)) < 1e-14
    assert abs(o[0, 0] - (7 + 28 - 28) / 7.0) < 1e-14


def test_constant_v():
    q, K = rand16(8, 128), rand16(2, 50, 128)
    v0 = rand16(2, 1, 128)
    V = np.repeat(v0, 50, axis=1)
    o, _ = oracle.attend(q, K, V)
    for h in range(8):
        assert np.abs(o[h] - v0[h // 4, 0].astype(np.float64)).max() < 1e-14


def test_output_in_convex_hull():
    q, K, V = rand16(8, 128), rand16(2, 64, 128), rand16(2, 64, 128)
    o, _ = oracle.attend(q, K, V)
    for h in range(8):
        v = V[h // 4].astype(np.float64)
        assert (o[h] <= v.max(axis=0) + 1e-14).all() and (o[h] >= v.min(axis=0) - 1e-14).all()


def test_permutation_invariance():
    q, K, V = rand16(4, 128), rand16(1, 200, 128), rand16(1, 200, 128)
    perm = RNG.permutation(200)
    o1, l1 = oracle.attend(q, K, V)
    o2, l2 = oracle.attend(q, np.ascontiguousarray(K[:, perm]), np.ascontiguousarray(V[:, perm]))
    assert np.abs(o1 - o2).max() < 1e-13 and np.abs(l1 - l2).max() < 1e-13


def test_score_shift_moves_lse_only():
    # keys K' = K + c*e_0 with q[0] = 1: every score moves by scale*c exactly (values chosen exact in fp16)
    q = rand16(1, 128)
    q[0, 0] = 1.0
    K = (RNG.integers(-8, 8, size=(1, 30, 128)) / 4.0).astype(np.float16)
    V = rand16(1, 30, 128)
    K2 = K.copy()
    K2[0, :, 0] += np.float16(2.0)
    o1, l1 = oracle.attend(q, K, V, scale=0.5)
    o2, l2 = oracle.attend(q, K2, V, scale=0.5)
    assert abs((l2[0] - l1[0]) - 1.0) < 1e-12
    assert np.abs(o1 - o2).max() < 1e-13


def test_scale_is_applied_before_softmax():
    q, K, V = rand16(2, 128), rand16(1, 40, 128), rand16(1, 40, 128)
    o_a, l_a = oracle.attend(q, K, V, scale=0.1)
    q2 = (q.astype(np.float32) * 2).astype(np.float16)  # exact doubling
    o_b, l_b = oracle.attend(q2, K, V, scale=0.05)
    assert np.abs(o_a - o_b).max() < 1e-13 and np.abs(l_a - l_b).max() < 1e-13
    # default scale is 1/sqrt(d)
    o_c, l_c = oracle.attend(q, K, V)
    o_d, l_d = oracle.attend(q, K, V, scale=1 / math.sqrt(128))
    assert np.array_equal(o_c, o_d) and np.array_equal(l_c, l_d)


# ---------------------------------------------------------------- GQA mapping -------------------
def test_gqa_mapping():
    Hq, Hkv, S = 8, 2, 33
    q1 = rand16(1, 128)
    q = np.repeat(q1, Hq, axis=0)
    K, V = rand16(Hkv, S, 128), rand16(Hkv, S, 128)
    o, lse = oracle.attend(q, K, V)
    # heads of one group with identical q give identical outputs; different groups differ
    for h in (1, 2, 3):
        assert np.array_equal(o[h], o[0]) and lse[h] == lse[0]
    for h in (5, 6, 7):
        assert np.array_equal(o[h], o[4])
    assert not np.array_equal(o[0], o[4])
    # perturbing kv head 1 leaves heads 0..3 bit-identical, changes heads 4..7
    K2, V2 = K.copy(), V.copy()
    K2[1] = rand16(S, 128)
    V2[1] = rand16(S, 128)
    o2, lse2 = oracle.attend(q, K2, V2)
    assert np.array_equal(o2[:4], o[:4]) and np.array_equal(lse2[:4], lse[:4])
    assert not np.array_equal(o2[4:], o[4:])


# ---------------------------------------------------------------- library routines --------------
@pytest.mark.parametrize("S", [1, 5, 257, 4096, 65536])
def test_against_numpy_scipy(S):
    from scipy.special import logsumexp, softmax
    Hq, Hkv = 8, 2
    q, K, V = rand16(Hq, 128), rand16(Hkv, S, 128), rand16(Hkv, S, 128)
    o, lse = oracle.attend(q, K, V)
    sc = 1 / math.sqrt(128)
    for h in range(Hq):
        s = sc * (K[h // 4].astype(np.float64) @ q[h].astype(np.float64))
        assert abs(lse[h] - logsumexp(s)) < 1e-12
        assert np.abs(o[h] - softmax(s) @ V[h // 4].astype(np.float64)).max() < 1e-12


def test_range_restriction_against_numpy():
    from scipy.special import logsumexp, softmax
    q, K, V = rand16(4, 128), rand16(1, 100, 128), rand16(1, 100, 128)
    o, lse = oracle.attend(q, K, V, t_begin=17, t_end=64)
    sc = 1 / math.sqrt(128)
    for h in range(4):
        s = sc * (K[0, 17:64].astype(np.float64) @ q[h].astype(np.float64))
        assert abs(lse[h] - logsumexp(s)) < 1e-12
        assert np.abs(o[h] - softmax(s) @ V[0, 17:64].astype(np.float64)).max() < 1e-12


def test_bruteforce_mpmath():
    import mpmath as mp
    mp.mp.dps = 40
    Hq, Hkv, S, d = 2, 1, 9, 16
    q, K, V = rand16(Hq, d, scale=2.0), rand16(Hkv, S, d, scale=2.0), rand16(Hkv, S, d)
    o, lse = oracle.attend(q, K, V, scale=0.3)
    for h in range(Hq):
        s = [mp.mpf("0.3") * sum(mp.mpf(float(q[h, i])) * mp.mpf(float(K[0, t, i])) for i in range(d))
             for t in range(S)]
        Z = sum(mp.e ** x for x in s)
        # note: oracle's scale is the double nearest 0.3, mp's is exact 0.3 -> 1e-16-relative difference
        assert abs(mp.mpf(lse[h]) - mp.log(Z)) < 1e-13
        for j in range(d):
            ref = sum(mp.e ** s[t] * mp.mpf(float(V[0, t, j])) for t in range(S)) / Z
            assert abs(mp.mpf(o[h, j]) - ref) < 1e-13


def test_peaked_softmax():
    # SURVEY 8(c) "peaked softmax": one key = 4*q -> score ~ 45, weight ~ 1, o ~ V[t*]
    S, tstar = 300, 123
    q = gen.gen_q(0, 0, 0, 4)
    K, V = gen.gen_k(0, 0, np.arange(S), 1), gen.gen_v(0, 0, np.arange(S), 1)
    K = K.copy()
    K[0, tstar] = (q[2].astype(np.float32) * 4).astype(np.float16)
    o, lse = oracle.attend(q, K, V)
    s = 4 * (q[2].astype(np.float64) @ q[2].astype(np.float64)) / math.sqrt(128)
    assert s > 30
    assert abs(lse[2] - s) < 1e-9
    assert np.abs(o[2] - V[0, tstar].astype(np.float64)).max() < 1e-9


# ---------------------------------------------------------------- golden values ------------------
def test_golden_t0():
    g = load_golden("appendix_b_t0.json")
    q = gen.gen_q(0, 0, 0, 8)
    K, V = gen.gen_k(0, 0, np.arange(5), 2), gen.gen_v(0, 0, np.arange(5), 2)
    tol = g["abs_tol"]
    o, lse = oracle.attend(q, K, V)
    assert np.abs(lse - g["lse"]).max() < tol
    assert np.abs(o[:, 0] - g["o_col0"]).max() < tol
    assert np.abs(o[:, 127] - g["o_col127"]).max() < tol
    op, lp = oracle.attend_ranges(q, K, V, 4)
    assert np.abs(lp[0] - g["lse_range0"]).max() < tol
    assert np.abs(lp[1] - g["lse_range1"]).max() < tol
    for h in range(8):  # 1-token range: o = V exactly
        assert np.array_equal(op[1, h], V[h // 4, 4].astype(np.float64))
    assert op[1, 0, 0] == g["range1_o_h0_first2"][0] and op[1, 0, 1] == g["range1_o_h0_first2"][1]
    m = g["mpmath_head5"]
    assert abs(lse[5] - m["lse"]) < 1e-13 and abs(o[5, 0] - m["o0"]) < 1e-14 and abs(o[5, 127] - m["o127"]) < 1e-14


def test_golden_cfg1():
    g = load_golden("appendix_b_cfg1.json")
    S = g["S"]
    q = gen.gen_q(0, 0, 0, 32)
    K, V = gen.gen_k(0, 0, np.arange(S), 8), gen.gen_v(0, 0, np.arange(S), 8)
    o, lse = oracle.attend(q, K, V)
    op, lp = oracle.attend_ranges(q, K, V, g["R"])
    rt = g["rel_tol"]

    def close(a, b, tol=rt):
        return abs(a - b) <= tol * max(1.0, abs(b)) + 5e-13  # golden values carry 13 significant digits

    for hs, e in g["heads"].items():
        h = int(hs)
        assert close(lse[h], e["lse"]) and close(lp[0, h], e["lse_r0"]) and close(lp[1, h], e["lse_r1"])
        assert close(o[h, 0], e["o0"]) and close(o[h, 64], e["o64"]) and close(o[h, 127], e["o127"])
    assert abs(lse.sum() - g["sum_lse"]) < 1e-9
    assert abs(o.sum() - g["sum_o"]) < 1e-11
    assert abs(np.abs(o).sum() - g["sum_abs_o"]) < 1e-9
    assert abs(np.abs(o).max() - g["max_abs_o"]) < 1e-8
    m = g["mpmath_head13"]
    assert abs(lse[13] - m["lse"]) < 2e-14 * 10 and abs(o[13, 0] - m["o0"]) < 1e-15 * 10
    assert abs(o[13, 64] - m["o64"]) < 1e-16 * 100 and abs(o[13, 127] - m["o127"]) < 1e-15 * 10
    om, lm = oracle.merge(op, lp)
    assert np.abs(om - o).max() < 1e-14 and np.abs(lm - lse).max() < 1e-13


def _gen_head(stream, g, pos):
    """one kv head [1][len(pos)][128] of request 0 / layer 0, generated in chunks to bound memory"""
    out = np.empty((1, len(pos), 128), np.float16)
    key = gen.stream_key(gen.SEED, stream)
    d = np.arange(128, dtype=np.uint64)[None, :]
    for a in range(0, len(pos), 65536):
        p = np.asarray(pos[a:a + 65536], dtype=np.uint64)[:, None]
        out[0, a:a + 65536] = gen.normal16(gen.hash64(key, gen.make_idx(0, 0, p, g, d)))
    return out


def test_golden_cfg4_ranges_and_one_full_head():
    """cfg 4 (S = 1,048,576): range-0 / range-31 partial lse of four heads, and the full 1M-token result
    of head 0 (the others would only repeat the same code path at 20 s apiece)."""
    g = load_golden("appendix_b_cfg4.json")
    R, S = g["R"], g["S"]
    q = gen.gen_q(0, 0, 0, 64)
    rt = g["rel_tol"]
    for hs, e in g["heads"].items():
        h = int(hs)
        kv = h // 8
        for j, key in ((0, "lse_range0"), (31, "lse_range31")):
            pos = np.arange(j * R, (j + 1) * R)
            K, V = _gen_head(gen.STREAM_K, kv, pos), _gen_head(gen.STREAM_V, kv, pos)
            _, lse = oracle.attend(q[h:h + 1], K, V)
            assert abs(lse[0] - e[key]) <= rt * abs(e[key]) + 5e-13
    pos = np.arange(S)
    K, V = _gen_head(gen.STREAM_K, 0, pos), _gen_head(gen.STREAM_V, 0, pos)
    o, lse = oracle.attend(q[0:1], K, V)
    e = g["heads"]["0"]
    assert abs(lse[0] - e["lse"]) <= rt * abs(e["lse"])
    assert abs(o[0, 0] - e["o0"]) <= 1e-9 * abs(e["o0"]) and abs(o[0, 127] - e["o127"]) <= 1e-9 * abs(e["o127"])
    assert abs(np.abs(o[0]).max() - e["max_abs_o"]) < 1e-7
    # and the paper's exactness claim at full scale: merge of the 32 range partials == unsplit
    op, lp = oracle.attend_ranges(q[0:1], K, V, R)
    om, lm = oracle.merge(op, lp)
    assert np.abs(om - o).max() < 1e-14 and abs(lm[0] - lse[0]) < 1e-12


def test_half_conversion_exhaustive():
    """Every fp16 bit pattern passes through the oracle's own half->double conversion unchanged
    (1-token context returns V exactly), compared with numpy's conversion."""
    pats = np.arange(65536, dtype=np.uint16).view(np.float16)
    q = np.zeros((1, 128), np.float16)
    K = np.zeros((1, 1, 128), np.float16)
    for a in range(0, 65536, 128):
        V = pats[a:a + 128].reshape(1, 1, 128).copy()
        o, lse = oracle.attend(q, K, V)
        assert np.array_equal(o[0], V[0, 0].astype(np.float64), equal_nan=True)
        assert lse[0] == 0.0
