"""Pins for oracle/wside.c and oracle/wside.py (the W-node stages around core attention).
Chosen so that a transposed operand, a dropped term, a wrong activation or a missing storage rounding fails one."""
import math

import numpy as np
import pytest

from kf_inputs import gen
from oracle import wside


def test_hand_example_and_operand_order():
    # x [1][3] = (1, 2, 3); W [2][3] = ((1, 0, -1), (2, 1, 0)): y = (1 - 3, 2 + 2) = (-2, 4).  W is [out][in]: a
    # transposed read of W would need a [3][2] matrix and cannot produce this.
    y = wside.linear(np.array([[1.0, 2.0, 3.0]]), np.array([[1.0, 0.0, -1.0], [2.0, 1.0, 0.0]]))
    assert y.tolist() == [[-2.0, 4.0]]
    # two rows of x: rows are independent
    y = wside.linear(np.array([[1.0, 0.0], [0.0, 1.0]]), np.array([[3.0, 5.0], [7.0, 11.0], [13.0, 17.0]]))
    assert y.tolist() == [[3.0, 7.0, 13.0], [5.0, 11.0, 17.0]]


def test_identity_and_one_hot_rows():
    rng = np.random.default_rng(1)
    x = rng.standard_normal((5, 64))
    assert np.array_equal(wside.linear(x, np.eye(64)), x)                 # identity weights: y = x exactly
    W = np.zeros((3, 64))
    W[0, 7] = 1.0
    W[1, 63] = -2.0
    W[2, 0] = 0.5                                                        # one-hot rows pick (and scale) columns
    y = wside.linear(x, W)
    assert np.array_equal(y[:, 0], x[:, 7]) and np.array_equal(y[:, 1], -2.0 * x[:, 63])
    assert np.array_equal(y[:, 2], 0.5 * x[:, 0])


def test_linearity_and_library_matmul():
    rng = np.random.default_rng(2)
    x1, x2 = rng.standard_normal((4, 256)), rng.standard_normal((4, 256))
    W = rng.standard_normal((96, 256))
    y = wside.linear(3.0 * x1 - x2, W)
    assert np.abs(y - (3.0 * wside.linear(x1, W) - wside.linear(x2, W))).max() < 1e-12
    assert np.abs(wside.linear(x1, W) - x1 @ W.T).max() < 1e-12          # special case: numpy's fp64 matmul
    # fp16 inputs are taken exactly
    xh = x1.astype(np.float16)
    assert np.abs(wside.linear(xh, W) - xh.astype(np.float64) @ W.T).max() < 1e-12


def test_swiglu_values():
    # silu(z) = z / (1 + e^-z):  silu(0) = 0;  silu(ln 3) = ln 3 * 3/4;  silu(-ln 3) = -ln 3 / 4;  silu(z) - silu(-z) = z
    l3 = math.log(3.0)
    h = wside.swiglu(np.array([0.0, l3, -l3, 2.0]), np.array([5.0, 2.0, 4.0, 1.0]))
    assert h[0] == 0.0
    assert abs(h[1] - l3 * 0.75 * 2.0) < 1e-15 and abs(h[2] + l3 * 0.25 * 4.0) < 1e-15
    z = np.linspace(-6, 6, 25)
    assert np.abs(wside.swiglu(z, np.ones(25)) - wside.swiglu(-z, np.ones(25)) - z).max() < 1e-14
    # the gate is the FIRST argument: swapping gate and up changes the result
    assert not np.allclose(wside.swiglu(np.array([1.0]), np.array([3.0])), wside.swiglu(np.array([3.0]), np.array([1.0])))


def test_project_splits_k_then_v_and_rounds_what_is_stored():
    rng = np.random.default_rng(3)
    x = rng.standard_normal((2, 128)).astype(np.float16)
    Wq = rng.standard_normal((256, 128)).astype(np.float16)
    Wkv = np.zeros((8, 128), np.float16)
    Wkv[:4, 0] = 1.0                                                      # K rows read x[:, 0]
    Wkv[4:, 1] = 1.0                                                      # V rows read x[:, 1]
    p = wside.project(x, Wq, Wkv)
    assert np.array_equal(p["k"], np.repeat(x[:, :1].astype(np.float64), 4, 1))
    assert np.array_equal(p["v"], np.repeat(x[:, 1:2].astype(np.float64), 4, 1))
    assert p["q16"].dtype == np.float16 and np.array_equal(p["q16"], p["q"].astype(np.float16))
    assert np.abs(p["q16"].astype(np.float64) - p["q"]).max() > 0        # storage rounding really happens


def test_post_attention_chain_by_hand():
    # hidden = 2, H_q*d = 2, ffn = 2; Wo = I; Wg = I; Wu = 2I; Wd = [[1, 1], [0, 1]]:
    # o = (ln 3, 0) -> y = o -> g = y, u = 2y -> h = (ln3 * 3/4 * 2 ln3, 0) -> x' = (h0 + h1, h1)
    l3 = np.float16(math.log(3.0)).astype(np.float64)                     # the fp16 copy of o is what W_O sees
    eye = np.eye(2)
    r = wside.post_attention(np.array([[math.log(3.0), 0.0]]), eye, eye, 2 * eye, np.array([[1.0, 1.0], [0.0, 1.0]]))
    h0 = l3 / (1 + math.exp(-l3)) * 2 * l3
    assert r["y"][0, 0] == l3 and r["y"][0, 1] == 0
    assert abs(r["h"][0, 0] - h0) < 1e-15 and r["h"][0, 1] == 0
    h16 = np.float16(h0).astype(np.float64)                               # h is stored as fp16 before the down projection
    assert r["x"].tolist() == [[h16, 0.0]]
    assert r["x16"].dtype == np.float16


def test_synthetic_weights_have_unit_gain_and_are_stateless():
    W = gen.gen_weight(gen.STREAM_WQ, 0, 256, 4096)
    assert W.shape == (256, 4096) and W.dtype == np.float16
    assert abs(float(W.astype(np.float64).std()) * 64.0 - 1.0) < 0.02     # N(0,1) * 2^-6
    assert gen.weight_shift(4096) == 6 and gen.weight_shift(14336) == 7 and gen.weight_shift(1024) == 5
    # element [n][k] depends on (stream, layer, n, k) only
    W2 = gen.gen_weight(gen.STREAM_WQ, 0, 8, 256)
    W3 = gen.gen_weight(gen.STREAM_WQ, 0, 256, 256)
    assert np.array_equal(W2, W3[:8]) and np.array_equal(W3[:, :256] * np.float16(4.0), W[:, :256] * np.float16(16.0))
    assert not np.array_equal(gen.gen_weight(gen.STREAM_WO, 0, 8, 256), W2)
    x = gen.gen_x(0, 3, 5, 256)
    assert x.shape == (3, 256) and not np.array_equal(x[0], x[1])
    y = wside.linear(gen.gen_x(0, 16, 0, 4096), W)
    assert 0.8 < y.std() < 1.2
