"""Host-side checks of the C ABI (no GPU): the library builds, loads, exports every symbol the header declares,
and its pure-host entry points (sizes, offsets, validation, error strings) behave as documented."""
import ctypes
import os
import re

import pytest

from paper_2606_29207_b200 import KFlume, KFlumeError, load_library, make_config
from paper_2606_29207_b200.binding import EXPORTS

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_functions():
    src = open(os.path.join(ROOT, "include", "kflume.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(kf_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported():
    lib = load_library()
    names = header_functions()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/kflume.h but not exported"
    assert sorted(EXPORTS) == names


def test_version_and_strerror():
    lib = load_library()
    assert lib.kf_version() == 220
    assert lib.kf_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4):
        assert lib.kf_strerror(code) not in (b"ok", b"unknown error")
    assert lib.kf_strerror(-99) == b"unknown error"


def test_pool_bytes_match_paper_byte_formula():
    # per token per layer 2 * H_kv * d_h * 2 B  -> pool = that * R * slots * L
    lib = load_library()
    c = make_config(32, 8, 16384, 16, 128, 9, 40, n_layers=4)
    assert lib.kf_pool_bytes(ctypes.byref(c)) == 2 * 8 * 128 * 2 * 16384 * 40 * 4
    assert lib.kf_workspace_bytes(ctypes.byref(c)) > 0
    # layout: [layer][slot][kv_head][token][128] fp16, V half after the K half
    half = lib.kf_pool_bytes(ctypes.byref(c)) // 2
    assert lib.kf_pool_offset(ctypes.byref(c), 0, 0, 0, 0, 0) == 0
    assert lib.kf_pool_offset(ctypes.byref(c), 0, 0, 0, 1, 0) == 256
    assert lib.kf_pool_offset(ctypes.byref(c), 0, 0, 1, 0, 0) == 256 * 16384
    assert lib.kf_pool_offset(ctypes.byref(c), 0, 1, 0, 0, 0) == 256 * 16384 * 8
    assert lib.kf_pool_offset(ctypes.byref(c), 1, 0, 0, 0, 0) == 256 * 16384 * 8 * 40
    assert lib.kf_pool_offset(ctypes.byref(c), 3, 39, 7, 16383, 1) == 2 * half - 256
    assert lib.kf_pool_offset(ctypes.byref(c), 4, 0, 0, 0, 0) == ctypes.c_size_t(-1).value


@pytest.mark.parametrize("kw", [dict(n_q_heads=30), dict(head_dim=64), dict(range_tokens=48), dict(n_partitions=65),
                                dict(n_partitions=0), dict(n_q_heads=128, n_kv_heads=8), dict(max_requests=0),
                                dict(softmax_scale=-1.0), dict(attend_impl=7)])
def test_invalid_configs_rejected(kw):
    lib = load_library()
    base = dict(n_q_heads=32, n_kv_heads=8, range_tokens=1024, n_partitions=2, max_requests=4,
                max_ranges_per_request=4, slots_per_partition=8)
    base.update(kw)
    c = make_config(**base)
    assert lib.kf_pool_bytes(ctypes.byref(c)) == 0 and lib.kf_workspace_bytes(ctypes.byref(c)) == 0
    h = ctypes.c_void_p()
    dummy = (ctypes.c_void_p * max(1, base["n_partitions"]))()
    assert lib.kf_create(ctypes.byref(h), ctypes.byref(c), dummy, ctypes.c_void_p(256), 1 << 30) == -1
    assert not h


def test_null_ctx_calls_return_einval():
    lib = load_library()
    assert lib.kf_token_boundary(None, None) == -1
    assert lib.kf_step_commit(None, None) == -1
    assert lib.kf_status(None, None) == -1
    assert lib.kf_destroy(None) == -1
    assert lib.kf_launch_count(None) == 0
    # the calls added in round 2 follow the same convention: an error code, never a crash
    assert lib.kf_layer_step(None, 0, None, None, None, None, None, None, None, None) == -1
    assert lib.kf_redirect_tails(None, None, None) == -1
    assert lib.kf_route_begins(None, None, None) == -1
    assert lib.kf_set_active_partitions(None, None, None) == -1
    assert lib.kf_step_graph_launch(None, None, None, None, None, None, None) == -1
    assert lib.kf_step_graph_seq(None, 0) == 0
    assert lib.kf_w_project_q(None, 0, None, 1, None, None) == -1
    assert lib.kf_attend_static(None, 0, None, None, None, None) == -1
    assert lib.kf_route_install_latency(None, 1, None, None, None) == -1
    assert lib.kf_wside_launch_count(None) == 0


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(KFlumeError):
        KFlume(make_config(32, 8, 1024, 2, 4, 4, 8))
