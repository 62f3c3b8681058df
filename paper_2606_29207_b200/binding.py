"""Thin ctypes binding of libkflume (include/kflume.h).  Argument marshalling only: every step of the path
runs in the CUDA kernels behind the C ABI.  PyTorch is used for device memory and streams, nothing else.

There is no CPU fallback: constructing a `KFlume` without a CUDA device (or without the built library) raises.
"""
from __future__ import annotations

import ctypes
from typing import Optional, Sequence

from . import build as _build

KF_OK, KF_EINVAL, KF_ESTATE, KF_ENOSPC, KF_ECUDA = 0, -1, -2, -3, -4
KF_IMPL_AUTO, KF_IMPL_SIMPLE, KF_IMPL_TMA = 0, 1, 2

EXPORTS = [
    "kf_version", "kf_strerror", "kf_last_cuda_error", "kf_pool_bytes", "kf_workspace_bytes", "kf_pool_offset",
    "kf_create", "kf_destroy", "kf_open_request", "kf_close_request", "kf_load_context", "kf_token_boundary",
    "kf_kv_append", "kf_partial_attend", "kf_merge_partials", "kf_attend", "kf_attend_static", "kf_step_commit", "kf_layer_step", "kf_layer_step_host",
    "kf_route_snapshot", "kf_status", "kf_plan_info", "kf_launch_count", "kf_worker_times",
    "kf_step_graph_create", "kf_step_graph_launch", "kf_step_graph_destroy", "kf_probe_read",
    "kf_step_graph_flags", "kf_step_graph_seq", "kf_step_graph_release", "kf_signal_roundtrip", "kf_route_install_latency",
    "kf_set_active_partitions", "kf_redirect_tails", "kf_route_begins", "kf_partition_state", "kf_set_active_requests",
    "kf_policy_bytes_per_token", "kf_policy_threshold", "kf_policy_initial_nodes", "kf_policy_step",
    "kf_wside_weight_bytes", "kf_wside_weight_offset", "kf_wside_workspace_bytes", "kf_wside_create", "kf_wside_destroy",
    "kf_wside_last_error", "kf_wside_launch_count", "kf_wside_set_sms", "kf_w_project_q", "kf_w_project_kv", "kf_w_post_attention",
    "kf_pipeline_step",
]
KF_W_Q, KF_W_KV, KF_W_O, KF_W_GATE, KF_W_UP, KF_W_DOWN = range(6)


class kf_config(ctypes.Structure):
    _fields_ = [
        ("n_q_heads", ctypes.c_int32), ("n_kv_heads", ctypes.c_int32), ("head_dim", ctypes.c_int32),
        ("n_layers", ctypes.c_int32), ("range_tokens", ctypes.c_int32), ("n_partitions", ctypes.c_int32),
        ("max_requests", ctypes.c_int32), ("max_ranges_per_request", ctypes.c_int32),
        ("slots_per_partition", ctypes.c_int32), ("softmax_scale", ctypes.c_float),
        ("attend_impl", ctypes.c_int32), ("min_tiles_per_worker", ctypes.c_int32),
        ("workers_per_sm", ctypes.c_int32), ("pipeline_stages", ctypes.c_int32),
        ("sched_first_pct", ctypes.c_int32), ("sched_decay_pct", ctypes.c_int32),
        ("plan_refresh_steps", ctypes.c_int32), ("kv_l2_policy", ctypes.c_int32),
        ("attend_sms", ctypes.c_int32), ("diagnostics", ctypes.c_int32),
    ]


class kf_wside_config(ctypes.Structure):
    _fields_ = [("hidden", ctypes.c_int32), ("n_q_heads", ctypes.c_int32), ("n_kv_heads", ctypes.c_int32),
                ("head_dim", ctypes.c_int32), ("ffn", ctypes.c_int32), ("n_layers", ctypes.c_int32),
                ("max_batch", ctypes.c_int32)]


class kf_policy_config(ctypes.Structure):
    _fields_ = [("beta_mem", ctypes.c_double), ("beta_slo", ctypes.c_double), ("gamma", ctypes.c_double),
                ("t_a_max_s", ctypes.c_double), ("bw_hbm", ctypes.c_double), ("c_kv_cap", ctypes.c_double),
                ("t_step_s", ctypes.c_double), ("t_prewarm_s", ctypes.c_double),
                ("n_kv_heads", ctypes.c_int32), ("head_dim", ctypes.c_int32), ("n_layers", ctypes.c_int32)]


class kf_policy_decision(ctypes.Structure):
    _fields_ = [("tau_fill", ctypes.c_double), ("want_prewarm", ctypes.c_int32), ("want_publish", ctypes.c_int32)]


class KFlumeError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libkflume: {msg} (code {code})")
        self.code = code


_lib = None


def load_library():
    """dlopen the in-tree libkflume.so (building it if sources are newer) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    L = ctypes.CDLL(_build.build())
    vp, i32, i64, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_size_t
    cfgp = ctypes.POINTER(kf_config)
    L.kf_version.restype = ctypes.c_int
    L.kf_strerror.argtypes, L.kf_strerror.restype = [ctypes.c_int], ctypes.c_char_p
    L.kf_last_cuda_error.argtypes, L.kf_last_cuda_error.restype = [vp], ctypes.c_char_p
    L.kf_pool_bytes.argtypes, L.kf_pool_bytes.restype = [cfgp], sz
    L.kf_workspace_bytes.argtypes, L.kf_workspace_bytes.restype = [cfgp], sz
    L.kf_pool_offset.argtypes, L.kf_pool_offset.restype = [cfgp, i32, i32, i32, i32, i32], sz
    L.kf_create.argtypes = [ctypes.POINTER(vp), cfgp, ctypes.POINTER(vp), vp, sz]
    L.kf_destroy.argtypes = [vp]
    L.kf_open_request.argtypes = [vp, i32, i32, vp]
    L.kf_close_request.argtypes = [vp, i32, vp]
    L.kf_load_context.argtypes = [vp, i32, i32, i32, i32, vp, vp, vp]
    L.kf_token_boundary.argtypes = [vp, vp]
    L.kf_kv_append.argtypes = [vp, i32, vp, vp, vp]
    L.kf_partial_attend.argtypes = [vp, i32, vp, ctypes.POINTER(ctypes.c_uint8), vp, vp, vp]
    L.kf_merge_partials.argtypes = [vp, vp, vp, vp, vp, vp]
    L.kf_attend.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp]
    L.kf_attend_static.argtypes = [vp, i32, vp, vp, vp, vp]
    L.kf_step_commit.argtypes = [vp, vp]
    L.kf_layer_step.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp, vp]
    L.kf_layer_step_host.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp]
    L.kf_route_snapshot.argtypes = [vp] + [ctypes.POINTER(i32)] * 6 + [vp]
    L.kf_status.argtypes = [vp, vp]
    L.kf_plan_info.argtypes = [vp, ctypes.POINTER(i32), vp]
    L.kf_launch_count.argtypes, L.kf_launch_count.restype = [vp], i64
    L.kf_worker_times.argtypes = [vp, ctypes.POINTER(i64), ctypes.POINTER(i32), vp]
    pp = ctypes.POINTER(vp)
    L.kf_step_graph_create.argtypes = [vp, i32, ctypes.POINTER(i32), i32, pp, pp, pp, pp, pp, vp, ctypes.POINTER(vp)]
    L.kf_step_graph_launch.argtypes = [vp, pp, pp, pp, pp, pp, vp]
    L.kf_step_graph_destroy.argtypes = [vp]
    L.kf_step_graph_flags.argtypes = [vp, vp, i32, vp]
    L.kf_step_graph_seq.argtypes, L.kf_step_graph_seq.restype = [vp, i32], ctypes.c_uint32
    L.kf_step_graph_release.argtypes = [vp, i32, ctypes.c_uint32, vp]
    L.kf_signal_roundtrip.argtypes = [vp, i32, vp, vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    L.kf_route_install_latency.argtypes = [vp, i32, vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    L.kf_set_active_partitions.argtypes = [vp, ctypes.POINTER(ctypes.c_uint8), vp]
    L.kf_redirect_tails.argtypes = [vp, ctypes.POINTER(ctypes.c_uint8), vp]
    L.kf_route_begins.argtypes = [vp, ctypes.POINTER(ctypes.c_int32), vp]
    L.kf_set_active_requests.argtypes = [vp, vp, vp]
    L.kf_partition_state.argtypes = [vp, ctypes.POINTER(i32), ctypes.POINTER(i64), ctypes.POINTER(i32), vp]
    pcp = ctypes.POINTER(kf_policy_config)
    u8p = ctypes.POINTER(ctypes.c_uint8)
    L.kf_policy_bytes_per_token.argtypes, L.kf_policy_bytes_per_token.restype = [pcp], ctypes.c_double
    L.kf_policy_threshold.argtypes, L.kf_policy_threshold.restype = [pcp], ctypes.c_double
    L.kf_policy_initial_nodes.argtypes, L.kf_policy_initial_nodes.restype = [pcp, ctypes.POINTER(i64), i32], i64
    L.kf_policy_step.argtypes = [pcp, i32, ctypes.POINTER(i64), ctypes.POINTER(i32), u8p, u8p,
                                 ctypes.POINTER(kf_policy_decision)]
    L.kf_probe_read.argtypes = [vp, vp, ctypes.POINTER(sz), vp]
    wcp = ctypes.POINTER(kf_wside_config)
    L.kf_wside_weight_bytes.argtypes, L.kf_wside_weight_bytes.restype = [wcp], sz
    L.kf_wside_weight_offset.argtypes, L.kf_wside_weight_offset.restype = [wcp, i32, i32], sz
    L.kf_wside_workspace_bytes.argtypes, L.kf_wside_workspace_bytes.restype = [wcp], sz
    L.kf_wside_create.argtypes = [ctypes.POINTER(vp), wcp, vp, vp, sz]
    L.kf_wside_destroy.argtypes = [vp]
    L.kf_wside_set_sms.argtypes = [vp, i32]
    L.kf_wside_last_error.argtypes, L.kf_wside_last_error.restype = [vp], ctypes.c_char_p
    L.kf_wside_launch_count.argtypes, L.kf_wside_launch_count.restype = [vp], i64
    L.kf_w_project_q.argtypes = [vp, i32, vp, i32, vp, vp]
    L.kf_w_project_kv.argtypes = [vp, i32, vp, i32, vp, vp, vp]
    L.kf_w_post_attention.argtypes = [vp, i32, vp, i32, vp, vp]
    L.kf_pipeline_step.argtypes = [vp, pp, i32, i32, ctypes.POINTER(i32), pp, pp, pp, pp, pp, pp, i32, vp, vp]
    for name in EXPORTS:
        if getattr(L, name).restype is None:
            getattr(L, name).restype = ctypes.c_int
    _lib = L
    return L


def make_config(n_q_heads, n_kv_heads, range_tokens, n_partitions, max_requests, max_ranges_per_request,
                slots_per_partition, n_layers=1, softmax_scale=0.0, attend_impl=KF_IMPL_AUTO,
                min_tiles_per_worker=0, head_dim=128, workers_per_sm=0, pipeline_stages=0, sched_first_pct=0,
                sched_decay_pct=0, plan_refresh_steps=0, kv_l2_policy=0, diagnostics=0, attend_sms=0) -> kf_config:
    c = kf_config()
    c.n_q_heads, c.n_kv_heads, c.head_dim, c.n_layers = n_q_heads, n_kv_heads, head_dim, n_layers
    c.range_tokens, c.n_partitions, c.max_requests = range_tokens, n_partitions, max_requests
    c.max_ranges_per_request, c.slots_per_partition = max_ranges_per_request, slots_per_partition
    c.softmax_scale, c.attend_impl, c.min_tiles_per_worker = softmax_scale, attend_impl, min_tiles_per_worker
    c.workers_per_sm, c.pipeline_stages = workers_per_sm, pipeline_stages
    c.sched_first_pct, c.sched_decay_pct = sched_first_pct, sched_decay_pct
    c.plan_refresh_steps = plan_refresh_steps
    c.kv_l2_policy = kv_l2_policy
    c.diagnostics = diagnostics
    c.attend_sms = attend_sms
    return c


def _ptr(t) -> ctypes.c_void_p:
    return ctypes.c_void_p(0 if t is None else t.data_ptr())


class KFlume:
    """One libkflume context plus the device memory it works on (allocated here with torch, owned by this object)."""

    def __init__(self, cfg: kf_config, device: str = "cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise KFlumeError(KF_ECUDA, "no CUDA device: libkflume has no CPU fallback")
        self.lib = load_library()
        self.cfg = cfg
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        pb = self.lib.kf_pool_bytes(ctypes.byref(cfg))
        wb = self.lib.kf_workspace_bytes(ctypes.byref(cfg))
        if pb == 0 or wb == 0:
            raise KFlumeError(KF_EINVAL, "invalid kf_config")
        self.pool_bytes, self.workspace_bytes = pb, wb
        self._pool_store = [torch.empty(pb + 1024, dtype=torch.uint8, device=self.device)
                            for _ in range(cfg.n_partitions)]
        self.pools = []
        for t in self._pool_store:
            off = (-t.data_ptr()) % 1024
            self.pools.append(t[off:off + pb])
        self._ws_store = torch.empty(wb + 256, dtype=torch.uint8, device=self.device)
        off = (-self._ws_store.data_ptr()) % 256
        self.workspace = self._ws_store[off:off + wb]
        arr = (ctypes.c_void_p * cfg.n_partitions)(*[p.data_ptr() for p in self.pools])
        h = ctypes.c_void_p()
        rc = self.lib.kf_create(ctypes.byref(h), ctypes.byref(cfg), arr, _ptr(self.workspace), wb)
        self.h = h
        if rc != KF_OK:
            msg = self.lib.kf_last_cuda_error(h).decode() if h else ""
            if h:
                self.lib.kf_destroy(h)
                self.h = None
            raise KFlumeError(rc, f"kf_create: {self.lib.kf_strerror(rc).decode()} {msg}")
        self.B, self.Hq, self.Hkv = cfg.max_requests, cfg.n_q_heads, cfg.n_kv_heads
        self.Jmax, self.P = cfg.max_ranges_per_request, cfg.n_partitions

    # ------------------------------------------------------------------------------------------------
    def close(self):
        if getattr(self, "h", None):
            self.torch.cuda.synchronize(self.device)
            self.lib.kf_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _stream(self, stream=None) -> ctypes.c_void_p:
        s = self.torch.cuda.current_stream(self.device) if stream is None else stream
        return ctypes.c_void_p(s.cuda_stream)

    def _check(self, rc: int, what: str):
        if rc != KF_OK:
            extra = self.lib.kf_last_cuda_error(self.h).decode() if rc == KF_ECUDA else ""
            raise KFlumeError(rc, f"{what}: {self.lib.kf_strerror(rc).decode()} {extra}")

    def _f16(self, t, shape):
        assert t.is_cuda and t.dtype == self.torch.float16 and t.is_contiguous() and tuple(t.shape) == tuple(shape), \
            (t.dtype, tuple(t.shape), tuple(shape))
        return _ptr(t)

    def _f32(self, t, shape):
        assert t.is_cuda and t.dtype == self.torch.float32 and t.is_contiguous() and tuple(t.shape) == tuple(shape), \
            (t.dtype, tuple(t.shape), tuple(shape))
        return _ptr(t)

    # ---- same names as the C ABI --------------------------------------------------------------------
    def open_request(self, req: int, n_tokens: int, stream=None):
        self._check(self.lib.kf_open_request(self.h, req, n_tokens, self._stream(stream)), "kf_open_request")

    def close_request(self, req: int, stream=None):
        self._check(self.lib.kf_close_request(self.h, req, self._stream(stream)), "kf_close_request")

    def load_context(self, layer: int, req: int, tok_begin: int, k, v, stream=None):
        n = k.shape[1]
        self._check(self.lib.kf_load_context(self.h, layer, req, tok_begin, n, self._f16(k, (self.Hkv, n, 128)),
                                             self._f16(v, (self.Hkv, n, 128)), self._stream(stream)),
                    "kf_load_context")

    def token_boundary(self, stream=None):
        self._check(self.lib.kf_token_boundary(self.h, self._stream(stream)), "kf_token_boundary")

    def kv_append(self, layer: int, k_new, v_new, stream=None):
        shp = (self.B, self.Hkv, 128)
        self._check(self.lib.kf_kv_append(self.h, layer, self._f16(k_new, shp), self._f16(v_new, shp),
                                          self._stream(stream)), "kf_kv_append")

    def partial_attend(self, layer: int, q, o_part, lse_part, partition_mask: Optional[Sequence[int]] = None,
                       stream=None):
        mask = None
        if partition_mask is not None:
            assert len(partition_mask) == self.P
            mask = (ctypes.c_uint8 * self.P)(*[1 if x else 0 for x in partition_mask])
        self._check(self.lib.kf_partial_attend(
            self.h, layer, self._f16(q, (self.B, self.Hq, 128)), mask,
            self._f32(o_part, (self.B, self.Jmax, self.Hq, 128)), self._f32(lse_part, (self.B, self.Jmax, self.Hq)),
            self._stream(stream)), "kf_partial_attend")

    def merge_partials(self, o_part, lse_part, o, lse, stream=None):
        self._check(self.lib.kf_merge_partials(
            self.h, self._f32(o_part, (self.B, self.Jmax, self.Hq, 128)),
            self._f32(lse_part, (self.B, self.Jmax, self.Hq)), self._f32(o, (self.B, self.Hq, 128)),
            self._f32(lse, (self.B, self.Hq)), self._stream(stream)), "kf_merge_partials")

    def attend(self, layer: int, q, o, lse, o_part=None, lse_part=None, stream=None):
        if o_part is not None:
            self._f32(o_part, (self.B, self.Jmax, self.Hq, 128))
            self._f32(lse_part, (self.B, self.Jmax, self.Hq))
        self._check(self.lib.kf_attend(self.h, layer, self._f16(q, (self.B, self.Hq, 128)),
                                       self._f32(o, (self.B, self.Hq, 128)), self._f32(lse, (self.B, self.Hq)),
                                       _ptr(o_part), _ptr(lse_part), self._stream(stream)), "kf_attend")

    def attend_static(self, layer: int, q, o, lse, stream=None):
        """kf_attend with the range partials in the library's own fixed device array: for callers that can neither pass
        scratch memory nor allocate it (see include/kflume.h).  Results equal attend(layer, q, o, lse) bit for bit."""
        rc = self.lib.kf_attend_static(self.h, layer, self._f16(q, (self.B, self.Hq, 128)),
                                       self._f32(o, (self.B, self.Hq, 128)), self._f32(lse, (self.B, self.Hq)),
                                       self._stream(stream))
        if rc != KF_OK:   # the size limit is reported as KF_EINVAL with the byte counts in the ctx's error text
            raise KFlumeError(rc, f"kf_attend_static: {self.lib.kf_strerror(rc).decode()} "
                                  f"{self.lib.kf_last_cuda_error(self.h).decode()}")

    def step_commit(self, stream=None):
        self._check(self.lib.kf_step_commit(self.h, self._stream(stream)), "kf_step_commit")

    def layer_step(self, layer: int, q, k_new, v_new, o, lse, o_part=None, lse_part=None, stream=None):
        if o_part is not None:
            self._f32(o_part, (self.B, self.Jmax, self.Hq, 128))
            self._f32(lse_part, (self.B, self.Jmax, self.Hq))
        shp = (self.B, self.Hkv, 128)
        self._check(self.lib.kf_layer_step(self.h, layer, self._f16(q, (self.B, self.Hq, 128)), self._f16(k_new, shp),
                                           self._f16(v_new, shp), self._f32(o, (self.B, self.Hq, 128)),
                                           self._f32(lse, (self.B, self.Hq)), _ptr(o_part), _ptr(lse_part),
                                           self._stream(stream)), "kf_layer_step")

    def layer_step_host(self, layer: int, q_host, k_new_host, v_new_host, o_host, lse_host, stream=None):
        for t in (q_host, k_new_host, v_new_host, o_host, lse_host):
            assert not t.is_cuda and t.is_contiguous()
        assert q_host.numel() == self.B * self.Hq * 128 and k_new_host.numel() == self.B * self.Hkv * 128
        assert o_host.numel() == self.B * self.Hq * 128 and o_host.dtype == self.torch.float32
        self._check(self.lib.kf_layer_step_host(self.h, layer, _ptr(q_host), _ptr(k_new_host), _ptr(v_new_host),
                                                _ptr(o_host), _ptr(lse_host), self._stream(stream)),
                    "kf_layer_step_host")

    def step_graph_create(self, layers: Sequence[int], q, k_new, v_new, o, lse, host_io: bool = False, stream=None):
        """kf_step_graph_create: q .. lse are lists (one tensor per layer-step).  Returns a StepGraph."""
        return StepGraph(self, layers, q, k_new, v_new, o, lse, host_io, stream)

    def probe_read(self, sink, stream=None) -> int:
        """kf_probe_read: stream all KV pools once (measurement aid); sink: 4-byte CUDA tensor.  Returns bytes read."""
        n = ctypes.c_size_t(0)
        self._check(self.lib.kf_probe_read(self.h, _ptr(sink), ctypes.byref(n), self._stream(stream)), "kf_probe_read")
        return int(n.value)

    def route_install_latency(self, iters: int, stream=None):
        """kf_route_install_latency: (enqueue_us, complete_us) medians of a route install issued from C."""
        q, c = ctypes.c_double(), ctypes.c_double()
        self._check(self.lib.kf_route_install_latency(self.h, iters, self._stream(stream), ctypes.byref(q),
                                                      ctypes.byref(c)), "kf_route_install_latency")
        return q.value, c.value

    def signal_roundtrip(self, iters: int, exec_stream, signal_stream):
        """kf_signal_roundtrip: (median_us, min_us) of gate release -> readiness flag seen by the host."""
        med, mn = ctypes.c_double(0), ctypes.c_double(0)
        self._check(self.lib.kf_signal_roundtrip(self.h, iters, ctypes.c_void_p(exec_stream.cuda_stream),
                                                 ctypes.c_void_p(signal_stream.cuda_stream), ctypes.byref(med),
                                                 ctypes.byref(mn)), "kf_signal_roundtrip")
        return med.value, mn.value

    def set_active_partitions(self, active: Sequence[int], stream=None):
        assert len(active) == self.P
        arr = (ctypes.c_uint8 * self.P)(*[1 if x else 0 for x in active])
        self._check(self.lib.kf_set_active_partitions(self.h, arr, self._stream(stream)), "kf_set_active_partitions")

    def redirect_tails(self, partitions: Sequence[int], stream=None):
        assert len(partitions) == self.P
        arr = (ctypes.c_uint8 * self.P)(*[1 if x else 0 for x in partitions])
        self._check(self.lib.kf_redirect_tails(self.h, arr, self._stream(stream)), "kf_redirect_tails")

    def set_active_requests(self, active=None, stream=None):
        """active: CUDA uint8 tensor [B] (non-zero = takes part in decode steps) or None = all."""
        if active is not None:
            assert active.is_cuda and active.dtype == self.torch.uint8 and active.numel() == self.B
        self._check(self.lib.kf_set_active_requests(self.h, _ptr(active), self._stream(stream)), "kf_set_active_requests")

    def partition_state(self, stream=None) -> dict:
        act, tok, tails = (ctypes.c_int32 * self.P)(), (ctypes.c_int64 * self.P)(), (ctypes.c_int32 * self.P)()
        self._check(self.lib.kf_partition_state(self.h, act, tok, tails, self._stream(stream)), "kf_partition_state")
        return {"active": list(act), "tokens": list(tok), "tails": list(tails)}

    def route_snapshot(self, stream=None) -> dict:
        i32 = ctypes.c_int32
        ln, nr = (i32 * self.B)(), (i32 * self.B)()
        part, slot = (i32 * (self.B * self.Jmax))(), (i32 * (self.B * self.Jmax))()
        fh, cur = (i32 * self.P)(), (i32 * 1)()
        self._check(self.lib.kf_route_snapshot(self.h, ln, nr, part, slot, fh, cur, self._stream(stream)),
                    "kf_route_snapshot")
        begin = (i32 * (self.B * self.Jmax))()
        self._check(self.lib.kf_route_begins(self.h, begin, self._stream(stream)), "kf_route_begins")
        J = self.Jmax
        return {"len": list(ln), "n_ranges": list(nr),
                "part": [list(part[r * J:(r + 1) * J]) for r in range(self.B)],
                "slot": [list(slot[r * J:(r + 1) * J]) for r in range(self.B)],
                "begin": [list(begin[r * J:(r + 1) * J]) for r in range(self.B)],
                "free_head": list(fh), "rr_cursor": cur[0]}

    def status(self, stream=None) -> int:
        return self.lib.kf_status(self.h, self._stream(stream))

    def plan_info(self, stream=None) -> dict:
        out = (ctypes.c_int32 * 8)()
        self._check(self.lib.kf_plan_info(self.h, out, self._stream(stream)), "kf_plan_info")
        keys = ["n_units", "n_tiles", "n_workers", "n_pieces", "n_entries", "tile_tokens", "max_workers", "pad"]
        return dict(zip(keys, list(out)))

    def worker_times(self, stream=None):
        """[(smid, t_start, t_first, t_end)] in ns for every worker of the last attend launch."""
        n = ctypes.c_int32(0)
        buf = (ctypes.c_int64 * (2048 * 4))()
        self._check(self.lib.kf_worker_times(self.h, buf, ctypes.byref(n), self._stream(stream)), "kf_worker_times")
        return [tuple(buf[4 * i:4 * i + 4]) for i in range(n.value)]

    def launch_count(self) -> int:
        return int(self.lib.kf_launch_count(self.h))

    def pool_offset(self, layer: int, slot: int, kv_head: int, token: int, is_v: bool) -> int:
        return int(self.lib.kf_pool_offset(ctypes.byref(self.cfg), layer, slot, kv_head, token, 1 if is_v else 0))


class StepGraph:
    """kf_graph handle: one decode step (token boundary, n x (append, attend), commit) as a static CUDA graph."""

    def __init__(self, kf: KFlume, layers, q, k_new, v_new, o, lse, host_io=False, stream=None):
        self.kf, self.n, self.host_io = kf, len(layers), bool(host_io)
        for lst in (q, k_new, v_new, o, lse):
            assert len(lst) == self.n
            for t in lst:
                assert t.is_contiguous() and t.is_cuda != self.host_io
        self._keep = (list(q), list(k_new), list(v_new), list(o), list(lse))  # bound buffers stay alive
        arr = (ctypes.c_int32 * self.n)(*layers)
        h = ctypes.c_void_p()
        kf._check(kf.lib.kf_step_graph_create(kf.h, self.n, arr, 1 if host_io else 0, *self._arrays(*self._keep),
                                              kf._stream(stream), ctypes.byref(h)), "kf_step_graph_create")
        self.h = h

    def _arrays(self, q, k_new, v_new, o, lse):
        return [(ctypes.c_void_p * self.n)(*[t.data_ptr() for t in lst]) for lst in (q, k_new, v_new, o, lse)]

    def launch(self, q=None, k_new=None, v_new=None, o=None, lse=None, stream=None):
        """One decode step.  Pass all five lists to re-bind the pointers (device tensors, or pinned host tensors for a
        host-io graph), or none to keep them."""
        if q is None:
            args = [None] * 5
        else:
            self._keep = (list(q), list(k_new), list(v_new), list(o), list(lse))
            args = self._arrays(*self._keep)
        self.kf._check(self.kf.lib.kf_step_graph_launch(self.h, *args, self.kf._stream(stream)), "kf_step_graph_launch")

    def flags(self, ready_host=None, gates: bool = False, stream=None):
        """kf_step_graph_flags: ready_host = pinned int32/uint32 CPU tensor [n] (or None); gates = wait before each
        layer-step until released.  Call before the first launch."""
        if ready_host is not None:
            assert not ready_host.is_cuda and ready_host.is_pinned() and ready_host.numel() == self.n
            assert ready_host.element_size() == 4 and ready_host.is_contiguous()
        self._ready = ready_host
        self.kf._check(self.kf.lib.kf_step_graph_flags(self.h, _ptr(ready_host), 1 if gates else 0,
                                                       self.kf._stream(stream)), "kf_step_graph_flags")

    def seq(self, layer_step: int) -> int:
        """Sequence number layer-step i carries in the NEXT launch."""
        return int(self.kf.lib.kf_step_graph_seq(self.h, layer_step))

    def release(self, layer_step: int, seq: int, signal_stream):
        """kf_step_graph_release on the DEDICATED signalling stream."""
        self.kf._check(self.kf.lib.kf_step_graph_release(self.h, layer_step, seq,
                                                         ctypes.c_void_p(signal_stream.cuda_stream)),
                       "kf_step_graph_release")

    def destroy(self):
        if getattr(self, "h", None) and self.kf.h:
            self.kf.torch.cuda.synchronize(self.kf.device)
            self.kf.lib.kf_step_graph_destroy(self.h)
        self.h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class Policy:
    """Algorithm 1 of the paper (kf_policy_*): host-side arithmetic only, usable without a GPU."""

    def __init__(self, **kw):
        self.lib = load_library()
        self.cfg = kf_policy_config(**kw)

    def bytes_per_token(self) -> float:
        return self.lib.kf_policy_bytes_per_token(ctypes.byref(self.cfg))

    def threshold(self) -> float:
        return self.lib.kf_policy_threshold(ctypes.byref(self.cfg))

    def initial_nodes(self, lengths: Sequence[int]) -> int:
        arr = (ctypes.c_int64 * len(lengths))(*lengths)
        return int(self.lib.kf_policy_initial_nodes(ctypes.byref(self.cfg), arr, len(lengths)))

    def step(self, tokens: Sequence[int], tails: Sequence[int], pending: Sequence[int], ready: Sequence[int]):
        P = len(tokens)
        out = (kf_policy_decision * P)()
        rc = self.lib.kf_policy_step(ctypes.byref(self.cfg), P, (ctypes.c_int64 * P)(*tokens),
                                     (ctypes.c_int32 * P)(*tails), (ctypes.c_uint8 * P)(*[1 if x else 0 for x in pending]),
                                     (ctypes.c_uint8 * P)(*[1 if x else 0 for x in ready]), out)
        if rc != KF_OK:
            raise KFlumeError(rc, "kf_policy_step: invalid argument")
        return [(d.tau_fill, bool(d.want_prewarm), bool(d.want_publish)) for d in out]


class WSide:
    """The W-node stages (kf_wside_*, kf_w_*): QKV projection, W_O and the SwiGLU FFN as tcgen05 GEMMs, plus the
    M-microbatch inter-layer pipeline (kf_pipeline_step).  Owns the weight and workspace buffers (torch)."""

    def __init__(self, hidden: int, n_q_heads: int, n_kv_heads: int, ffn: int, n_layers: int = 1, max_batch: int = 128,
                 device: str = "cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise KFlumeError(KF_ECUDA, "no CUDA device: libkflume has no CPU fallback")
        self.lib, self.torch = load_library(), torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        c = kf_wside_config(hidden, n_q_heads, n_kv_heads, 128, ffn, n_layers, max_batch)
        self.cfg = c
        wb, sb = self.lib.kf_wside_weight_bytes(ctypes.byref(c)), self.lib.kf_wside_workspace_bytes(ctypes.byref(c))
        if wb == 0 or sb == 0:
            raise KFlumeError(KF_EINVAL, "invalid kf_wside_config")
        self._w_store = torch.empty(wb + 1024, dtype=torch.uint8, device=self.device)
        off = (-self._w_store.data_ptr()) % 1024
        self.weights = self._w_store[off:off + wb]
        self._s_store = torch.empty(sb + 256, dtype=torch.uint8, device=self.device)
        off = (-self._s_store.data_ptr()) % 256
        self.workspace = self._s_store[off:off + sb]
        h = ctypes.c_void_p()
        rc = self.lib.kf_wside_create(ctypes.byref(h), ctypes.byref(c), _ptr(self.weights), _ptr(self.workspace), sb)
        self.h = h
        if rc != KF_OK:
            msg = self.lib.kf_wside_last_error(h).decode() if h else ""
            if h:
                self.lib.kf_wside_destroy(h)
                self.h = None
            raise KFlumeError(rc, f"kf_wside_create: {self.lib.kf_strerror(rc).decode()} {msg}")
        self.hidden, self.Hq, self.Hkv, self.ffn, self.L = hidden, n_q_heads, n_kv_heads, ffn, n_layers

    def shape(self, which: int):
        qd, kvd = self.Hq * 128, self.Hkv * 128
        return {KF_W_Q: (qd, self.hidden), KF_W_KV: (2 * kvd, self.hidden), KF_W_O: (self.hidden, qd),
                KF_W_GATE: (self.ffn, self.hidden), KF_W_UP: (self.ffn, self.hidden),
                KF_W_DOWN: (self.hidden, self.ffn)}[which]

    def weight(self, layer: int, which: int):
        """fp16 view [out_features][in_features] of one weight matrix inside the weight buffer (write into it)."""
        off = self.lib.kf_wside_weight_offset(ctypes.byref(self.cfg), layer, which)
        n, k = self.shape(which)
        return self.weights[off:off + n * k * 2].view(self.torch.float16).view(n, k)

    def _stream(self, stream=None):
        s = self.torch.cuda.current_stream(self.device) if stream is None else stream
        return ctypes.c_void_p(s.cuda_stream)

    def _check(self, rc, what):
        if rc != KF_OK:
            extra = self.lib.kf_wside_last_error(self.h).decode() if rc == KF_ECUDA else ""
            raise KFlumeError(rc, f"{what}: {self.lib.kf_strerror(rc).decode()} {extra}")

    def project_q(self, layer, x, q, stream=None):
        B = x.shape[0]
        assert x.is_cuda and x.dtype == self.torch.float16 and x.is_contiguous() and x.shape == (B, self.hidden)
        assert q.is_cuda and q.dtype == self.torch.float16 and q.is_contiguous() and q.numel() == B * self.Hq * 128
        self._check(self.lib.kf_w_project_q(self.h, layer, _ptr(x), B, _ptr(q), self._stream(stream)), "kf_w_project_q")

    def project_kv(self, layer, x, k_new, v_new, stream=None):
        B = x.shape[0]
        assert x.is_cuda and x.dtype == self.torch.float16 and x.is_contiguous() and x.shape == (B, self.hidden)
        for t in (k_new, v_new):
            assert t.is_cuda and t.dtype == self.torch.float16 and t.is_contiguous() and t.numel() == B * self.Hkv * 128
        self._check(self.lib.kf_w_project_kv(self.h, layer, _ptr(x), B, _ptr(k_new), _ptr(v_new), self._stream(stream)),
                    "kf_w_project_kv")

    def post_attention(self, layer, o, x_next, stream=None):
        B = o.shape[0]
        assert o.is_cuda and o.dtype == self.torch.float32 and o.is_contiguous() and o.numel() == B * self.Hq * 128
        assert x_next.is_cuda and x_next.dtype == self.torch.float16 and x_next.is_contiguous()
        assert x_next.shape == (B, self.hidden)
        self._check(self.lib.kf_w_post_attention(self.h, layer, _ptr(o), B, _ptr(x_next), self._stream(stream)),
                    "kf_w_post_attention")

    def pipeline_step(self, kfs, layers, x, q, k_new, v_new, o, lse, pipelined, w_stream, a_stream):
        """kf_pipeline_step: kfs = list of KFlume (one per microbatch); x .. lse = lists of CUDA tensors."""
        M = len(kfs)
        arr = lambda lst: (ctypes.c_void_p * M)(*[t.data_ptr() for t in lst])   # noqa: E731
        ctxs = (ctypes.c_void_p * M)(*[k.h.value for k in kfs])
        la = (ctypes.c_int32 * len(layers))(*layers)
        self._check(self.lib.kf_pipeline_step(self.h, ctxs, M, len(layers), la, arr(x), arr(q), arr(k_new), arr(v_new),
                                              arr(o), arr(lse), 1 if pipelined else 0,
                                              ctypes.c_void_p(w_stream.cuda_stream), ctypes.c_void_p(a_stream.cuda_stream)),
                    "kf_pipeline_step")

    def set_sms(self, n_sms: int):
        """kf_wside_set_sms: CTAs of the persistent GEMM grid (0 = all SMs)."""
        self._check(self.lib.kf_wside_set_sms(self.h, n_sms), "kf_wside_set_sms")

    def launch_count(self) -> int:
        return int(self.lib.kf_wside_launch_count(self.h))

    def close(self):
        if getattr(self, "h", None):
            self.torch.cuda.synchronize(self.device)
            self.lib.kf_wside_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
