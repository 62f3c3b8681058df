"""Drive libkflume with the seeded synthetic workloads of kf_inputs (tests, bench.py, smoke).

Product-side helper: it only calls the C ABI (through binding.KFlume) and the shared input generator; it never
touches oracle/.  State preparation follows SURVEY.md 8(d): "context S" = S tokens resident at attend time, the
current token included -> open S-1 tokens, token_boundary, kv_append(position S-1), attend over len+1 = S.
"""
from __future__ import annotations

from typing import List, Optional

from kf_inputs import gen, gen_device
from kf_inputs.workloads import Workload

from .binding import (KF_IMPL_AUTO, KF_W_DOWN, KF_W_GATE, KF_W_KV, KF_W_O, KF_W_Q, KF_W_UP, KFlume, WSide,
                      make_config)


class Session:
    def __init__(self, wl: Workload, impl: int = KF_IMPL_AUTO, n_layers_phys: Optional[int] = None,
                 steps: Optional[int] = None, min_tiles: int = 0, device: str = "cuda:0", softmax_scale: float = 0.0,
                 slack_slots: int = 0, slack_ranges: int = 0, **tuning):
        import torch
        self.torch = torch
        self.wl = wl
        self.steps = wl.n_steps if steps is None else steps
        self.L_phys = wl.n_layers if n_layers_phys is None else n_layers_phys
        self.len0: List[int] = [s - 1 for s in wl.contexts]      # tokens resident before step 0
        cfg = make_config(wl.n_q_heads, wl.n_kv_heads, wl.range_tokens, wl.n_partitions, wl.batch,
                          wl.max_ranges(self.steps) + slack_ranges, wl.slots_per_partition(self.steps) + slack_slots,
                          n_layers=self.L_phys, softmax_scale=softmax_scale, attend_impl=impl,
                          min_tiles_per_worker=min_tiles, **tuning)
        self.kf = KFlume(cfg, device)
        self.device = self.kf.device
        B, Hq, Hkv = wl.batch, wl.n_q_heads, wl.n_kv_heads
        self.o = torch.zeros((B, Hq, 128), dtype=torch.float32, device=self.device)
        self.lse = torch.zeros((B, Hq), dtype=torch.float32, device=self.device)
        self.o_part = torch.zeros((B, self.kf.Jmax, Hq, 128), dtype=torch.float32, device=self.device)
        self.lse_part = torch.zeros((B, self.kf.Jmax, Hq), dtype=torch.float32, device=self.device)
        self._len0_dev = torch.tensor(self.len0, dtype=torch.int32, device=self.device)
        self.step = 0

    # ---- state preparation --------------------------------------------------------------------------
    def open_all(self):
        for r, n in enumerate(self.len0):
            self.kf.open_request(r, n)

    def load_all(self, chunk_tokens: int = 65536, layers: Optional[List[int]] = None):
        """Fill the routed pools with the generator's K/V for positions [0, len0_r) of every physical layer."""
        wl = self.wl
        layers = list(range(self.L_phys)) if layers is None else layers
        kbuf = self.torch.empty((wl.n_kv_heads, chunk_tokens, 128), dtype=self.torch.float16, device=self.device)
        vbuf = self.torch.empty_like(kbuf)
        for layer in layers:
            for r, n in enumerate(self.len0):
                for t0 in range(0, n, chunk_tokens):
                    m = min(chunk_tokens, n - t0)
                    k = kbuf.view(-1)[: wl.n_kv_heads * m * 128].view(wl.n_kv_heads, m, 128)
                    v = vbuf.view(-1)[: wl.n_kv_heads * m * 128].view(wl.n_kv_heads, m, 128)
                    gen_device.fill(gen.STREAM_K, layer, r, t0, m, wl.n_kv_heads, out=k, seed=wl.seed)
                    gen_device.fill(gen.STREAM_V, layer, r, t0, m, wl.n_kv_heads, out=v, seed=wl.seed)
                    self.kf.load_context(layer, r, t0, k, v)
        self.torch.cuda.synchronize(self.device)

    def prepare(self):
        self.open_all()
        self.load_all()

    # ---- per-step inputs (generator values keyed by PHYSICAL layer; SURVEY 8(d) cfg-5 aliasing) --------
    def q_for(self, layer_phys: int, step: int):
        pos = self.torch.full((self.wl.batch,), step, dtype=self.torch.int32, device=self.device)
        return gen_device.fill_rows(gen.STREAM_Q, layer_phys, pos, self.wl.n_q_heads, seed=self.wl.seed)

    def kv_new_for(self, layer_phys: int, step: int):
        pos = self._len0_dev + step
        k = gen_device.fill_rows(gen.STREAM_K, layer_phys, pos, self.wl.n_kv_heads, seed=self.wl.seed)
        v = gen_device.fill_rows(gen.STREAM_V, layer_phys, pos, self.wl.n_kv_heads, seed=self.wl.seed)
        return k, v

    # ---- one layer-step through the C ABI -------------------------------------------------------------
    def layer_step(self, layer: int, q, k_new, v_new, fused: bool = True, want_partials: bool = False,
                   one_launch: bool = False):
        kf = self.kf
        if one_launch:          # kf_layer_step: append + attend + merge in ONE launch (what the step graph replays)
            if want_partials:
                kf.layer_step(layer, q, k_new, v_new, self.o, self.lse, self.o_part, self.lse_part)
            else:
                kf.layer_step(layer, q, k_new, v_new, self.o, self.lse)
            return
        kf.kv_append(layer, k_new, v_new)
        if fused:
            if want_partials:
                kf.attend(layer, q, self.o, self.lse, self.o_part, self.lse_part)
            else:
                kf.attend(layer, q, self.o, self.lse)
        else:
            kf.partial_attend(layer, q, self.o_part, self.lse_part)
            kf.merge_partials(self.o_part, self.lse_part, self.o, self.lse)

    def close(self):
        self.kf.close()


W_STREAMS = {KF_W_Q: gen.STREAM_WQ, KF_W_KV: gen.STREAM_WKV, KF_W_O: gen.STREAM_WO, KF_W_GATE: gen.STREAM_WGATE,
             KF_W_UP: gen.STREAM_WUP, KF_W_DOWN: gen.STREAM_WDOWN}


def make_wside(hidden: int, n_q_heads: int, n_kv_heads: int, ffn: int, n_layers: int = 1, max_batch: int = 128,
               device: str = "cuda:0", seed: int = gen.SEED) -> WSide:
    """A WSide whose weight buffer holds the seeded synthetic weights of kf_inputs (random-init stand-ins for the
    Llama-3.1 weights of PAPER.md:288): matrix `which` of layer l = gen.gen_weight(W_STREAMS[which], l, ...)."""
    w = WSide(hidden, n_q_heads, n_kv_heads, ffn, n_layers, max_batch, device)
    for layer in range(n_layers):
        for which, stream in W_STREAMS.items():
            n, k = w.shape(which)
            gen_device.fill_weight(stream, layer, n, k, out=w.weight(layer, which), seed=seed)
    w.torch.cuda.synchronize(w.device)
    return w


def pipeline_attend_sms(kv_bytes: int, weight_bytes: int, n_sms: int = 148) -> int:
    """SM budget of the attend kernels (kf_config.attend_sms) when kf_pipeline_step overlaps them with the W-side GEMMs on
    ONE GPU; the GEMMs get the rest (kf_wside_set_sms(n_sms - result)).  Both sides stream from the same HBM, so the SMs
    are split by the bytes each side has to move per (layer, microbatch), a little in favour of the GEMMs (they need
    more SMs per byte/s than the attend kernel, which saturates HBM from ~100 SMs), and clamped to the range in which
    the sweep of profiles/r02c_pipeline.md found every optimum: 68..116, in steps of 4."""
    share = kv_bytes / float(kv_bytes + weight_bytes)
    sms = int(round(0.8 * n_sms * share / 4.0)) * 4
    return max(68, min(116, sms))
