"""Oracle of the W-node stages around core attention -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

``wside.c`` holds the arithmetic (the triple-loop contraction and SwiGLU, fp64).  This module strings it into the two
W-side stages of the paper's pipeline model:

  T_p  proj(x)          q = x Wq^T ;  (k_new, v_new) = x Wkv^T                    (PAPER.md:143 step 1; Q first, :252)
  T_f  post(o)          y = o Wo^T ;  h = silu(y Wg^T) * (y Wu^T) ;  x' = h Wd^T    (PAPER.md:147 step 5, :254)

The paper's tensors are FP16 (Llama-3.1-8B-Instruct with real weights; north_star: fp16 q/K/V), so every
tensor that the method STORES between two kernels -- q, k_new, v_new, the fp16 copy of o that feeds W_O, y, h, x' -- is
rounded to binary16 here as well (reading 25); everything inside a contraction is fp64.  No residual
connections, norms or rotary embedding: the row of SURVEY 8(f) asks for the GEMM stages and their timing, and the
weights are synthetic (reading 26).
"""
from __future__ import annotations

import ctypes

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(_build.build())
        dp, i64 = ctypes.POINTER(ctypes.c_double), ctypes.c_int64
        L.kfo_linear.argtypes = [dp, dp, i64, i64, i64, dp]
        L.kfo_linear.restype = ctypes.c_int
        L.kfo_swiglu.argtypes = [dp, dp, i64, dp]
        L.kfo_swiglu.restype = ctypes.c_int
        _lib = L
    return _lib


def _d(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))      # fp16 -> fp64 is exact


def _p(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def linear(x, w):
    """y[b][n] = sum_k x[b][k] * w[n][k] in fp64.  x [B][K], w [N][K] (any float dtype; converted exactly)."""
    x, w = _d(x), _d(w)
    B, K = x.shape
    N, K2 = w.shape
    assert K == K2
    y = np.empty((B, N), dtype=np.float64)
    if lib().kfo_linear(_p(x), _p(w), B, N, K, _p(y)):
        raise RuntimeError("kfo_linear failed")
    return y


def swiglu(g, u):
    g, u = _d(g), _d(u)
    assert g.shape == u.shape
    h = np.empty_like(g)
    if lib().kfo_swiglu(_p(g), _p(u), g.size, _p(h)):
        raise RuntimeError("kfo_swiglu failed")
    return h


def f16(a):
    """The method's storage precision: round to IEEE binary16 (round-to-nearest-even), returned as fp16."""
    return np.asarray(a, dtype=np.float64).astype(np.float16)


def project(x, Wq, Wkv):
    """T_p.  x [B][hidden] fp16; Wq [H_q*d][hidden], Wkv [2*H_kv*d][hidden] fp16 (K rows first, then V rows).
    Returns {"q", "k", "v"}: fp64 values before storage rounding, and {"q16", "k16", "v16"}: what is stored."""
    q = linear(x, Wq)
    kv = linear(x, Wkv)
    n = Wkv.shape[0] // 2
    out = {"q": q, "k": kv[:, :n], "v": kv[:, n:]}
    out.update({k + "16": f16(v) for k, v in list(out.items())})
    return out


def post_attention(o, Wo, Wg, Wu, Wd):
    """T_f.  o [B][H_q*d] (the merged attention output, any float dtype); Wo [hidden][H_q*d]; Wg, Wu [ffn][hidden];
    Wd [hidden][ffn].  Every stored tensor is rounded to fp16 before it feeds the next contraction.
    Returns {"y", "h", "x"} (fp64, before storage rounding) and {"y16", "h16", "x16"}."""
    o16 = f16(o)
    y = linear(o16, Wo)
    y16 = f16(y)
    h = swiglu(linear(y16, Wg), linear(y16, Wu))
    h16 = f16(h)
    x = linear(h16, Wd)
    return {"y": y, "h": h, "x": x, "y16": y16, "h16": h16, "x16": f16(x), "o16": o16}
