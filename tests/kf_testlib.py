"""Shared helpers of the GPU parity tests: oracle evaluation on host copies of the seeded inputs and the
tolerance gates of BASELINE.json's north_star (reading 12)."""
import numpy as np

import oracle
from kf_inputs import gen, gen_device

O_ABS_TOL = 2e-3          # max |o - o*|                                  (north_star)
LSE_REL_TOL = 1e-4        # |lse - lse*| <= 1e-4 * max(1, |lse*|)         (north_star + reading 12 guard)
O_SMELL_REL = 1.5e-3      # scale-free bug-smell gate: max|o - o*| <= 1.5e-3 * max|o*| + 2e-6  (P is fp16 in PV)


def check_close(o, lse, o_ref, lse_ref, what=""):
    o, lse = np.asarray(o, np.float64), np.asarray(lse, np.float64)
    assert np.isfinite(o).all() and np.isfinite(lse).all(), f"{what}: non-finite output"
    eo = np.abs(o - o_ref).max()
    el = (np.abs(lse - lse_ref) / np.maximum(1.0, np.abs(lse_ref))).max()
    assert eo <= O_ABS_TOL, f"{what}: max|o-o*| = {eo:.3e} > {O_ABS_TOL}"
    assert el <= LSE_REL_TOL, f"{what}: rel lse err = {el:.3e} > {LSE_REL_TOL}"
    smell = O_SMELL_REL * np.abs(o_ref).max() + 2e-6
    assert eo <= smell, f"{what}: max|o-o*| = {eo:.3e} exceeds the scale-free gate {smell:.3e}"
    return eo, el


def host_kv(wl, layer, req, n_tokens, heads=None, from_device=True):
    """K, V [H_kv][n_tokens][128] fp16 on the host for positions [0, n_tokens) -- from the device twin of the
    generator for big contexts (checked bit-exact against gen.py in test_gpu_generator), else numpy."""
    Hkv = wl.n_kv_heads
    if from_device and n_tokens > 4096:
        k = gen_device.fill(gen.STREAM_K, layer, req, 0, n_tokens, Hkv, seed=wl.seed).cpu().numpy()
        v = gen_device.fill(gen.STREAM_V, layer, req, 0, n_tokens, Hkv, seed=wl.seed).cpu().numpy()
    else:
        pos = np.arange(n_tokens)
        k, v = gen.gen_k(layer, req, pos, Hkv, wl.seed), gen.gen_v(layer, req, pos, Hkv, wl.seed)
    return k, v


def oracle_request(wl, layer, req, step, n_tokens, heads=None, scale=None, ranges=False, K=None, V=None):
    """Oracle (o*, lse*) of request `req` at decode step `step` over n_tokens tokens, for the given query heads."""
    q = gen.gen_q(layer, req, step, wl.n_q_heads, wl.seed)
    if K is None:
        K, V = host_kv(wl, layer, req, n_tokens)
    if heads is None:
        # all heads: ONE call on the full [H_q] / [H_kv] tensors, so the oracle's own GQA mapping (query head h reads KV
        # head h / G) is the one under test, not a restatement of it here
        o, lse = oracle.attend(q, K, V, scale)
        if not ranges:
            return o, lse
        op, lp = oracle.attend_ranges(q, K, V, wl.range_tokens, scale)
        return o, lse, op, lp
    G = wl.group
    heads = list(heads)
    o = np.zeros((len(heads), 128))
    lse = np.zeros(len(heads))
    op = lp = None
    if ranges:
        J = -(-n_tokens // wl.range_tokens)
        op, lp = np.zeros((J, len(heads), 128)), np.zeros((J, len(heads)))
    for i, h in enumerate(heads):
        g = h // G
        qq, kk, vv = q[h:h + 1], K[g:g + 1], V[g:g + 1]
        oo, ll = oracle.attend(qq, kk, vv, scale)
        o[i], lse[i] = oo[0], ll[0]
        if ranges:
            a, b = oracle.attend_ranges(qq, kk, vv, wl.range_tokens, scale)
            op[:, i], lp[:, i] = a[:, 0], b[:, 0]
    return (o, lse, op, lp) if ranges else (o, lse)
