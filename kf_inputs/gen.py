"""Seeded, stateless synthetic-input generator (host / numpy side).

This module holds NO arithmetic of the method (no attention, no softmax, no routing):
it only produces the synthetic q / K / V values and the per-request context lengths that
stand in for the paper's workloads (PAPER.md:343 trace, :288 model activations), following
the recipe of SURVEY.md Appendix A.  Both the CPU oracle's tests and the CUDA path's tests
draw inputs from here (and from the device twin in ``gen_cuda.cu`` which must be bit-identical).

Recipe (all uint64 arithmetic wraps):
    mix64(z): z ^= z>>30; z *= 0xBF58476D1CE4E5B9; z ^= z>>27; z *= 0x94D049BB133111EB; z ^= z>>31
    key(seed, stream) = mix64(seed XOR stream*0xD1B54A32D192ED03)
    hash(key, idx)    = mix64(key + (idx+1)*0x9E3779B97F4A7C15)   # idx-th splitmix64 output
    normal16(x)       = fp16_rn( fp32(sum of the 8 bytes of x - 1020) * c ),  c = fp32 bits 0x3B9CC4BF
    idx(layer, req, pos, head, dim) = dim | head<<7 | pos<<14 | req<<38 | layer<<54
    streams: q=1 (pos field = decode step), K=2, V=3, cfg-3 lengths=0x33, cfg-5 lengths=0x55
    W-side stages: hidden state x=4 (pos field = decode step), weights Wq=0x10, Wkv=0x11, Wo=0x12,
    Wgate=0x13, Wup=0x14, Wdown=0x15: element [n][k] of a weight matrix [out_features][in_features] is
    normal16(hash(key, idx(layer, 0, pos=n, head=k>>7, dim=k&127))) * 2^-s with 2^-s ~ 1/sqrt(in_features)
    (an exact power-of-two scaling in fp16), so y = x W^T has unit variance for unit-variance x.
"""
from __future__ import annotations

import numpy as np

SEED = 260629207
STREAM_Q, STREAM_K, STREAM_V = 1, 2, 3
STREAM_LEN_CFG3, STREAM_LEN_CFG5 = 0x33, 0x55
STREAM_X = 4
STREAM_WQ, STREAM_WKV, STREAM_WO, STREAM_WGATE, STREAM_WUP, STREAM_WDOWN = 0x10, 0x11, 0x12, 0x13, 0x14, 0x15

_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_GOLD = np.uint64(0x9E3779B97F4A7C15)
_STREAM_MUL = np.uint64(0xD1B54A32D192ED03)
# c = 1/sqrt(8*(256^2-1)/12): Irwin-Hall of 8 bytes -> unit variance.  Fixed fp32 bit pattern.
_C32 = np.array([0x3B9CC4BF], dtype=np.uint32).view(np.float32)[0]


def mix64(z):
    z = np.asarray(z, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = z ^ (z >> np.uint64(30))
        z = z * _M1
        z = z ^ (z >> np.uint64(27))
        z = z * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def stream_key(seed: int, stream: int) -> np.uint64:
    with np.errstate(over="ignore"):
        return mix64(np.uint64(seed) ^ (np.uint64(stream) * _STREAM_MUL))


def hash64(key, idx):
    idx = np.asarray(idx, dtype=np.uint64)
    with np.errstate(over="ignore"):
        return mix64(np.uint64(key) + (idx + np.uint64(1)) * _GOLD)


def byte_sum(x):
    """Sum of the 8 bytes of each uint64 (0..2040)."""
    x = np.ascontiguousarray(np.asarray(x, dtype=np.uint64))
    return x.view(np.uint8).reshape(x.shape + (8,)).sum(axis=-1, dtype=np.int32)


def normal16(x):
    """uint64 hash -> fp16 approximately N(0,1) (|z| <= 4.88)."""
    s = (byte_sum(x) - 1020).astype(np.float32)
    return (s * _C32).astype(np.float16)


def make_idx(layer, req, pos, head, dim):
    a = [np.asarray(v, dtype=np.uint64) for v in (layer, req, pos, head, dim)]
    layer, req, pos, head, dim = a
    return (dim | (head << np.uint64(7)) | (pos << np.uint64(14))
            | (req << np.uint64(38)) | (layer << np.uint64(54)))


def tensor(stream: int, layer: int, req: int, pos, heads: int, seed: int = SEED,
           head_dim: int = 128) -> np.ndarray:
    """fp16 values [heads][len(pos)][head_dim] of one stream for positions ``pos``."""
    pos = np.atleast_1d(np.asarray(pos, dtype=np.uint64))
    key = stream_key(seed, stream)
    h = np.arange(heads, dtype=np.uint64)[:, None, None]
    p = pos[None, :, None]
    d = np.arange(head_dim, dtype=np.uint64)[None, None, :]
    return normal16(hash64(key, make_idx(layer, req, p, h, d)))


def gen_q(layer: int, req: int, step: int, n_q_heads: int, seed: int = SEED) -> np.ndarray:
    """q[H_q][128] fp16 of request ``req`` at decode step ``step``."""
    return tensor(STREAM_Q, layer, req, [step], n_q_heads, seed)[:, 0, :]


def gen_k(layer: int, req: int, pos, n_kv_heads: int, seed: int = SEED) -> np.ndarray:
    """K[H_kv][len(pos)][128] fp16 for logical token positions ``pos``."""
    return tensor(STREAM_K, layer, req, pos, n_kv_heads, seed)


def gen_v(layer: int, req: int, pos, n_kv_heads: int, seed: int = SEED) -> np.ndarray:
    return tensor(STREAM_V, layer, req, pos, n_kv_heads, seed)


def weight_shift(in_features: int) -> int:
    """s with 2^-s the power of two nearest to 1/sqrt(in_features) from below in log2 (4096 -> 6, 14336 -> 7)."""
    return int(round(0.5 * np.log2(in_features)))


def gen_weight(stream: int, layer: int, n_out: int, n_in: int, seed: int = SEED) -> np.ndarray:
    """Synthetic fp16 weight matrix [n_out][n_in] (n_in a multiple of 128) of one W-side stream."""
    assert n_in % 128 == 0
    t = tensor(stream, layer, 0, np.arange(n_out), n_in // 128, seed)            # [n_in/128][n_out][128]
    w = np.ascontiguousarray(t.transpose(1, 0, 2)).reshape(n_out, n_in)
    return (w.astype(np.float32) * np.float32(2.0 ** -weight_shift(n_in))).astype(np.float16)   # exact


def gen_x(layer: int, batch: int, step: int, hidden: int, seed: int = SEED) -> np.ndarray:
    """Hidden state x[batch][hidden] fp16 entering layer `layer` at decode step `step` (row r = request r)."""
    return np.stack([tensor(STREAM_X, layer, r, [step], hidden // 128, seed)[:, 0, :].reshape(hidden)
                     for r in range(batch)])
