"""ctypes wrapper of libkfgen.so (gen_cuda.cu): the device twin of gen.py.  torch is used only for the
output tensors and the current stream."""
from __future__ import annotations

import ctypes
import os
import subprocess

from . import gen

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "gen_cuda.cu")
LIB = os.path.join(HERE, "libkfgen.so")
_lib = None


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = [os.environ.get("NVCC", "nvcc"), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17",
           "-lineinfo", "-Xcompiler", "-fPIC", "-shared", "-o", tmp, SRC]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.kfgen_fill.argtypes = [ctypes.c_uint64, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int64,
                                 ctypes.c_int64, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
        L.kfgen_fill.restype = ctypes.c_int
        L.kfgen_fill_rows.argtypes = [ctypes.c_uint64, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_int,
                                      ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
        L.kfgen_fill_rows.restype = ctypes.c_int
        _lib = L
    return _lib


def _stream():
    import torch
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def fill(stream_id: int, layer: int, req: int, pos_begin: int, n_pos: int, heads: int, out=None,
         seed: int = gen.SEED):
    """fp16 CUDA tensor [heads][n_pos][128] of one stream (K=2, V=3, q=1)."""
    import torch
    if out is None:
        out = torch.empty((heads, n_pos, 128), dtype=torch.float16, device="cuda")
    assert out.is_cuda and out.dtype == torch.float16 and out.is_contiguous() and out.numel() >= heads * n_pos * 128
    rc = lib().kfgen_fill(seed, stream_id, layer, req, pos_begin, n_pos, heads, ctypes.c_void_p(out.data_ptr()),
                          _stream())
    if rc:
        raise RuntimeError(f"kfgen_fill: cudaError {rc}")
    return out


def fill_rows(stream_id: int, layer: int, pos, heads: int, out=None, seed: int = gen.SEED):
    """fp16 CUDA tensor [B][heads][128]: row r = request r at position pos[r] (int32 CUDA tensor; <0 skips)."""
    import torch
    assert pos.is_cuda and pos.dtype == torch.int32 and pos.is_contiguous()
    B = pos.numel()
    if out is None:
        out = torch.zeros((B, heads, 128), dtype=torch.float16, device="cuda")
    assert out.is_cuda and out.dtype == torch.float16 and out.is_contiguous()
    rc = lib().kfgen_fill_rows(seed, stream_id, layer, ctypes.c_void_p(pos.data_ptr()), B, heads,
                               ctypes.c_void_p(out.data_ptr()), _stream())
    if rc:
        raise RuntimeError(f"kfgen_fill_rows: cudaError {rc}")
    return out


def fill_weight(stream_id: int, layer: int, n_out: int, n_in: int, out=None, seed: int = gen.SEED):
    """Device twin of gen.gen_weight: fp16 CUDA tensor [n_out][n_in]."""
    import torch
    assert n_in % 128 == 0
    t = fill(stream_id, layer, 0, 0, n_out, n_in // 128, seed=seed)               # [n_in/128][n_out][128]
    w = t.permute(1, 0, 2).reshape(n_out, n_in) * (2.0 ** -gen.weight_shift(n_in))   # power of two: exact in fp16
    if out is None:
        return w.contiguous()
    out.copy_(w)
    return out


def fill_x(layer: int, batch: int, step: int, hidden: int, seed: int = gen.SEED):
    """Device twin of gen.gen_x: fp16 CUDA tensor [batch][hidden]."""
    import torch
    pos = torch.full((batch,), step, dtype=torch.int32, device="cuda")
    return fill_rows(gen.STREAM_X, layer, pos, hidden // 128, seed=seed).reshape(batch, hidden)
