"""CPU oracle for the KernelFlume hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It shares nothing with ``paper_2606_29207_b200`` (the CUDA path) and
imports nothing from it.

* ``attention.c``  -- fp64 softmax attention (whole request / one token range) and LSE merge
  (PAPER.md:81, :145-147, :254).
* ``routing.py``   -- integer model of the routing table, slot allocation and append positions
  (PAPER.md:149, :159-161, :173, :240).
"""
from __future__ import annotations

import ctypes
import math

import numpy as np

from . import build as _build
from .routing import RoutingModel  # noqa: F401

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(_build.build())
        u16p = ctypes.POINTER(ctypes.c_uint16)
        dp = ctypes.POINTER(ctypes.c_double)
        L.kfo_attend_head.argtypes = [u16p, u16p, u16p, ctypes.c_int64, ctypes.c_int64, ctypes.c_int,
                                      ctypes.c_double, dp, dp]
        L.kfo_attend_head.restype = ctypes.c_int
        L.kfo_attend_request.argtypes = [u16p, u16p, u16p, ctypes.c_int, ctypes.c_int, ctypes.c_int64,
                                         ctypes.c_int64, ctypes.c_int64, ctypes.c_int, ctypes.c_double,
                                         dp, dp, ctypes.c_int]
        L.kfo_attend_request.restype = ctypes.c_int
        L.kfo_merge_head.argtypes = [dp, dp, ctypes.c_int, ctypes.c_int, dp, dp]
        L.kfo_merge_head.restype = ctypes.c_int
        L.kfo_num_threads.restype = ctypes.c_int
        _lib = L
    return _lib


def default_scale(head_dim: int) -> float:
    """DESIGN.md reading 1: softmax scale = 1/sqrt(head_dim)."""
    return 1.0 / math.sqrt(head_dim)


def _u16(a: np.ndarray):
    assert a.dtype == np.float16 and a.flags.c_contiguous
    return a.view(np.uint16).ctypes.data_as(ctypes.POINTER(ctypes.c_uint16))


def _f16c(a) -> np.ndarray:
    a = np.asarray(a)
    if a.dtype != np.float16:
        raise TypeError("oracle inputs are fp16 (the method's storage type, PAPER.md:234)")
    return np.ascontiguousarray(a)


def attend(q, K, V, scale=None, t_begin=0, t_end=None, n_threads=0):
    """Attention of one request over tokens [t_begin, t_end).

    q [H_q][d] fp16;  K, V [H_kv][S][d] fp16  ->  (o [H_q][d] float64, lse [H_q] float64).
    ``t_begin=0, t_end=S`` is the unpartitioned definition; a sub-interval is one token range's partial.
    """
    q, K, V = _f16c(q), _f16c(K), _f16c(V)
    Hq, d = q.shape
    Hkv, S, d2 = K.shape
    assert d2 == d and V.shape == K.shape
    if t_end is None:
        t_end = S
    assert 0 <= t_begin < t_end <= S, "empty or out-of-range token interval"
    if scale is None:
        scale = default_scale(d)
    o = np.empty((Hq, d), dtype=np.float64)
    lse = np.empty((Hq,), dtype=np.float64)
    dp = ctypes.POINTER(ctypes.c_double)
    rc = lib().kfo_attend_request(_u16(q), _u16(K), _u16(V), Hq, Hkv, S, t_begin, t_end, d, float(scale),
                                  o.ctypes.data_as(dp), lse.ctypes.data_as(dp), int(n_threads))
    if rc:
        raise RuntimeError(f"kfo_attend_request failed: {rc}")
    return o, lse


def attend_ranges(q, K, V, range_tokens, scale=None, n_threads=0):
    """Per-range partials of one request: ranges j = [jR, min((j+1)R, S)).
    Returns (o_part [J][H_q][d], lse_part [J][H_q])."""
    S = K.shape[1]
    J = -(-S // range_tokens)
    o = np.empty((J,) + q.shape, dtype=np.float64)
    lse = np.empty((J, q.shape[0]), dtype=np.float64)
    for j in range(J):
        o[j], lse[j] = attend(q, K, V, scale, j * range_tokens, min((j + 1) * range_tokens, S), n_threads)
    return o, lse


def merge(o_part, lse_part):
    """LSE merge of partials: o_part [J][H][d], lse_part [J][H] -> (o [H][d], lse [H])."""
    o_part = np.ascontiguousarray(o_part, dtype=np.float64)
    lse_part = np.ascontiguousarray(lse_part, dtype=np.float64)
    J, H, d = o_part.shape
    assert lse_part.shape == (J, H)
    o = np.empty((H, d), dtype=np.float64)
    lse = np.empty((H,), dtype=np.float64)
    dp = ctypes.POINTER(ctypes.c_double)
    for h in range(H):
        oj = np.ascontiguousarray(o_part[:, h, :])
        lj = np.ascontiguousarray(lse_part[:, h])
        out_l = ctypes.c_double()
        rc = lib().kfo_merge_head(lj.ctypes.data_as(dp), oj.ctypes.data_as(dp), J, d,
                                  o[h].ctypes.data_as(dp), ctypes.byref(out_l))
        if rc:
            raise RuntimeError(f"kfo_merge_head failed: {rc}")
        lse[h] = out_l.value
    return o, lse


def num_threads() -> int:
    return int(lib().kfo_num_threads())
