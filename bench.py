#!/usr/bin/env python
"""bench.py -- decode core-attention HBM GB/s and us per layer-step (BASELINE.json `metric`) on B200.

A "step" is one pass of the whole hot path over one batch of synthetic input:
    kf_token_boundary -> per layer { kf_kv_append + kf_attend (split-KV attention + fused LSE merge) } -> kf_step_commit
(each layer-step is ONE launch, kf_layer_step: the append rides in the attend kernel)
so the contexts grow by one token per step exactly as in decoding.  Headline workload: cfg3 (configs[2] of
BASELINE.json: B=16, Llama-3.1-8B shape, log-normal contexts with median 80K, 32K ranges over 8 partitions) -- the
configuration the north_star target ">= 80% of peak HBM bandwidth at >= 32K context" is quoted on and the stand-in for
the paper's serving trace.  The same process then measures the other BASELINE configs (cfg1, cfg2, cfg4, cfg5) and
reports them as sub-records under "workloads" of the ONE JSON line (`--only` skips them; `--workload X` makes X the
headline).  For the single-layer configs a second, STATIC protocol (load S-1 tokens, boundary, append,
then repeat append + attend WITHOUT committing, so every repetition sees exactly the stated context) is reported
beside the growing-context loop.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--only] [--impl ours|reference]

N > 1 (torchrun): every rank runs an independent batch of the same recipe (seed + rank): the path shards over
independent requests with no data-path collective -> "scaling": "weak"; NCCL is used only for the barrier and the
max-over-ranks of the device time.
"""
from __future__ import annotations

import argparse
import gc
import hashlib
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "decode_core_attention_hbm_gbps"
UNIT = "GB/s"
NOMINAL_PEAK_GBS = 8000.0        # BASELINE.json's "~8 TB/s" denominator (context)
FALLBACK_PEAK_GBS = 6650.0       # B200_PROFILING.md fallback if MEASURED_PEAKS.json is absent
SUB_WORKLOADS = ["cfg1", "cfg2", "cfg4", "cfg5"]
# steps / warm-up / end-to-end steps of the sub-records (the headline takes --steps / --warmup)
SUB_STEPS = {"cfg1": (200, 10, 50), "cfg2": (100, 10, 50), "cfg3": (100, 10, 40), "cfg4": (60, 6, 30),
             "cfg5": (8, 3, 3)}

# dram__bytes_read.sum + dram__bytes_write.sum per kf_attend launch from the committed `ncu --set full` captures.
# A capture is only valid for the kernel sources it was taken from: `rev` is kernel_rev() at capture time, and the
# line carries `traffic` only when the running sources hash to the same value and no tuning flag is set.
NCU_TRAFFIC = {
    # workload: (bytes per launch, committed summary, kernel_rev at capture time)
    "cfg1": (16982400, "profiles/r02c_attend_full_cfg1.md", "a39d3ecfd9ff"),
    "cfg2": (1086072536, "profiles/r02c_attend_full_cfg2.md", "a39d3ecfd9ff"),
    "cfg3": (4782946188, "profiles/r02c_attend_full_cfg3.md", "a39d3ecfd9ff"),
    "cfg4": (4306954112, "profiles/r02c_attend_full_cfg4.md", "a39d3ecfd9ff"),
    "cfg5": (37122581380, "profiles/r02c_attend_full_cfg5.md", "a39d3ecfd9ff"),
    "fig10_q64kv8_b32_s32k": (4311526756, "profiles/r02c_attend_full_fig10_q64kv8_b32_s32k.md", "a39d3ecfd9ff"),
}


def kernel_rev():
    """Short hash of the sources of the dominant kernel: ties an ncu capture to the code it was taken from."""
    h = hashlib.sha256()
    for f in ("kf_attend_tma.cu", "kf_merge.cuh", "kf_common.cuh"):
        with open(os.path.join(ROOT, "paper_2606_29207_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:12]


def traffic_record(wl_name, args):
    cap = NCU_TRAFFIC.get(wl_name)
    if cap is None:
        return None, "no committed ncu capture for this workload"
    nbytes, src, rev = cap
    if args.attend_impl == 1 or args.min_tiles or args.kv_l2_policy or args.no_graph or args.workers_per_sm or args.stages:
        return None, f"{src}: not applicable (non-default --attend-impl / --min-tiles / --kv-l2-policy / --no-graph)"
    if rev != kernel_rev():
        return None, f"{src}: stale (captured at kernel_rev {rev}, running {kernel_rev()})"
    return nbytes, f"{src} (ncu --set full, committed; kernel_rev {rev})"


def load_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    except Exception:
        return FALLBACK_PEAK_GBS, "fallback (B200_PROFILING.md)"


# ---------------------------------------------------------------------------------------------------------
def algorithmic_bytes(wl, lens_before, n_layers):
    """Bytes the method must move in one step: per layer, every context token's
    K and V rows (2*H_kv*128*2 B) + q read + appended K/V rows read and written + outputs written +
    range partials written and re-read for requests with more than one range."""
    per_tok = wl.kv_bytes_per_token()
    B, Hq, Hkv, R = wl.batch, wl.n_q_heads, wl.n_kv_heads, wl.range_tokens
    kv = sum((n + 1) * per_tok for n in lens_before)
    q = B * Hq * 128 * 2
    app = 2 * (2 * B * Hkv * 128 * 2)
    out = B * Hq * (128 + 1) * 4
    part = 0
    for n in lens_before:
        J = -(-(n + 1) // R)
        if J > 1:
            part += 2 * J * Hq * (128 + 1) * 4
    return n_layers * (kv + q + app + out + part), n_layers * kv


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.rows, self.proc, self.gpu = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def mark(self):
        return time.perf_counter()

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        time.sleep(0.06)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.06] or [r for (_, r) in self.rows[-3:]]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0]))
                mx = float(f[1])
                for n, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------------
# The CPU oracle, timed as it stands on a bounded sample of the workload.  Shared by the `cpu_baseline` leg of our
# arm and by `--impl reference`, so both time THE SAME sample (the only places bench.py may execute oracle/).
def _host_kv(wl, r, n, have_gpu):
    import numpy as np
    from kf_inputs import gen
    if have_gpu:
        from kf_inputs import gen_device
        K = gen_device.fill(gen.STREAM_K, 0, r, 0, n, wl.n_kv_heads, seed=wl.seed).cpu().numpy()
        V = gen_device.fill(gen.STREAM_V, 0, r, 0, n, wl.n_kv_heads, seed=wl.seed).cpu().numpy()
        return K, V
    pos = np.arange(n)
    return gen.gen_k(0, r, pos, wl.n_kv_heads, wl.seed), gen.gen_v(0, r, pos, wl.n_kv_heads, wl.seed)


def oracle_sample(wl, lens_before, budget_s, have_gpu):
    """Pick the sample: the shortest requests of the batch (all query heads, layer 0) until ~budget_s of oracle work,
    estimated from a 2048-token probe; a single request that is too long is cut to a prefix.  Returns
    ([(request, n_tokens)], host K/V per entry, description)."""
    import oracle
    from kf_inputs import gen
    order = sorted(range(wl.batch), key=lambda r: lens_before[r])
    r0 = order[0]
    n0 = min(2048, lens_before[r0] + 1)
    K, V = _host_kv(wl, r0, n0, have_gpu)
    q = gen.gen_q(0, r0, 0, wl.n_q_heads, wl.seed)
    t = time.perf_counter()
    oracle.attend(q, K, V)
    rate = n0 / max(time.perf_counter() - t, 1e-6)          # context tokens / s (all heads)
    if not have_gpu:                                         # numpy generates ~2M elements/s: keep the sample small
        budget_s = min(budget_s, 65536 / rate)
    chosen, tok = [], 0
    for r in order:
        n = lens_before[r] + 1
        if chosen and (tok + n) / rate > budget_s:
            break
        chosen.append((r, n))
        tok += n
    if tok / rate > 2 * budget_s:                            # a single huge request: a prefix of its tokens
        chosen = [(chosen[0][0], max(256, int(rate * budget_s)))]
    data = [_host_kv(wl, r, n, have_gpu) for r, n in chosen]
    full = all(n == lens_before[r] + 1 for r, n in chosen)
    desc = (f"{wl.name} layer 0: requests {[r for r, _ in chosen]} "
            f"({sum(n for _, n in chosen)} context tokens{'' if full else ', PREFIX of the request'}, "
            f"all {wl.n_q_heads} query heads), oracle.attend fp64")
    return chosen, data, desc


def oracle_run(wl, chosen, data, step, n_threads=0):
    """One timed pass of the oracle over the sample (n_threads = 0: the oracle's default, all host cores).
    Returns (seconds, {request: (o*, lse*)})."""
    import oracle
    from kf_inputs import gen
    qs = [gen.gen_q(0, r, step, wl.n_q_heads, wl.seed) for r, _ in chosen]
    out = {}
    t = time.perf_counter()
    for (r, n), (K, V), q in zip(chosen, data, qs):
        out[r] = oracle.attend(q, K, V, n_threads=n_threads)
    return time.perf_counter() - t, out


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, timed on the host cores; every step is one pass over the same
    bounded sample the `cpu_baseline` leg of our arm uses (sized so that the whole run ends within a few minutes)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    from kf_inputs import workloads
    try:
        import torch
        have_gpu = torch.cuda.is_available()
    except Exception:
        have_gpu = False
    wl = workloads.by_name(args.workload)
    lens = [s - 1 for s in wl.contexts]
    n_steps = max(1, args.warmup + args.steps)
    chosen, data, desc = oracle_sample(wl, lens, min(15.0, 150.0 / n_steps), have_gpu)
    times = []
    for step in range(n_steps):
        dt, _ = oracle_run(wl, chosen, data, step)
        if step >= args.warmup:
            times.append(dt)
    dt = sum(times) / len(times)
    val = sum(n for _, n in chosen) * wl.kv_bytes_per_token() / dt / 1e9
    sample = desc + ", one pass per step"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "note": wl.note, "sample": sample},
            "sample": sample,
            "cpu_baseline": {"value": val, "unit": UNIT, "kind": "oracle", "cores": oracle.num_threads(), "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_route_install(args):
    """--route-install: one JSON line with signalling_record()."""
    import torch
    print(json.dumps(signalling_record(torch.device("cuda:0"), args.workload)))
    return 0


def signalling_record(dev, workload="cfg3"):
    """Latency of a scale event (kf_set_active_partitions, the paper's route install: 7.2 us on its
    CPU) and of kf_token_boundary with a kept / a rebuilt work plan.  Medians; one JSON line."""
    import statistics
    import torch
    from kf_inputs import workloads
    from paper_2606_29207_b200.workload import Session
    wl = workloads.by_name(workload)
    P = wl.n_partitions

    def event_us(fn):
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        t0 = time.perf_counter()
        fn()
        t1 = time.perf_counter()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) * 1e3, (t1 - t0) * 1e6

    out = {"mode": "route-install", "workload": wl.name, "n_partitions": P}
    for key, refresh in (("kept_plan", 0), ("rebuilt_plan", 1)):
        ses = Session(wl, n_layers_phys=1, steps=400, slack_slots=4, plan_refresh_steps=refresh)
        ses.open_all()                                   # routes only: pool contents do not matter here
        kf = ses.kf
        kf.token_boundary()
        if key == "kept_plan":
            ev, host = [], []
            for i in range(200):
                mask = [1] * P
                mask[i % P] = i % 2
                if not any(mask):
                    mask[0] = 1
                e, h = event_us(lambda: kf.set_active_partitions(mask))
                ev.append(e)
                host.append(h)
            kf.set_active_partitions([1] * P)
            out["set_active_event_us"] = statistics.median(ev)
            out["set_active_host_enqueue_us"] = statistics.median(host)
            # the same install issued from C inside the library (no ctypes, no torch stream look-up in the way)
            out["route_install_c_enqueue_us"], out["route_install_c_complete_us"] = kf.route_install_latency(2000)
        ev = []
        for _ in range(60):
            ev.append(event_us(kf.token_boundary)[0])
            kf.step_commit()
        out[f"token_boundary_{key}_event_us"] = statistics.median(ev)
        if key == "kept_plan":
            # graph progress signalling: gate release on the signalling stream -> ReadValue32-style wait
            # inside a running graph -> WriteValue32-style readiness flag -> seen by the spinning host thread
            med, mn = kf.signal_roundtrip(2000, torch.cuda.Stream(), torch.cuda.Stream())
            out["signal_roundtrip_us_median"], out["signal_roundtrip_us_min"] = med, mn
        assert kf.status() == 0
        ses.close()
    e = []
    for _ in range(60):
        e.append(event_us(lambda: None)[0])
    out["empty_event_pair_us"] = statistics.median(e)
    out["paper_route_install_us"] = 7.2          # PAPER.md:308 (its CPU routing loop; context, another machine)
    return out



def pipeline_cases(cases, sms_list, n_layers, want_parity=True):
    """W-side stages + M = 2 inter-layer kernel pipelining on ONE B200 (PAPER.md:252-280,
    Fig. 11): for each workload (two microbatches of B_mu requests at context S, Llama-3.1-8B shape, synthetic weights)
    measure T_p (Q + K/V projection), T_f (W_O + SwiGLU FFN), T_A (append + attend, as a function of the attend
    kernel's SM budget), the serial and the pipelined step, and compare the measured ratio with the paper's model
    G_pipe = (T_p + T_A + T_f) / max(T_p + T_f, T_A).  sms_list: attend SM budgets to try; None = the one
    `workload.pipeline_attend_sms` picks from the byte counts.  After the timed replays of a case ONE fresh pipelined step
    (layer 0) is compared with the oracle chain.  Returns the dict `--pipeline` prints."""
    import statistics
    import torch
    from kf_inputs import gen_device, workloads
    from kf_inputs.workloads import Workload
    from paper_2606_29207_b200.workload import Session, make_wside, pipeline_attend_sms

    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    hidden, Hq, Hkv, ffn = 4096, 32, 8, 14336
    Lw = 2                                           # physical weight layers (436 MB each >> L2), aliased
    w = make_wside(hidden, Hq, Hkv, ffn, n_layers=Lw, max_batch=128)
    weight_bytes_layer = sum(2 * a * b for a, b in (w.shape(i) for i in range(6)))
    peak, peak_src = load_peak()
    ws, as_ = torch.cuda.Stream(dev), torch.cuda.Stream(dev)

    def graph_us(fn, reps=12, inner=8):
        """Median device time of one fn(i), measured on replays of a CUDA graph that holds `inner` calls (the C-ABI
        calls are capturable; a replay takes the host launch cost out of the measurement)."""
        fn(0)
        ws.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=ws):
            for i in range(inner):
                fn(i)
        ts = []
        for i in range(3 + reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(ws)
            g.replay()
            b.record(ws)
            if i >= 3:
                ts.append((a, b))
        torch.cuda.synchronize(dev)
        del g
        return statistics.median(x.elapsed_time(y) for x, y in ts) * 1e3 / inner

    rows = []
    sms_arg = sms_list
    for (Bm, S) in cases:
        R, P = 8192, 4
        rec = {"B_mu": Bm, "seq": S, "microbatches": 2, "layers_per_step": n_layers}
        best = None
        # without a sweep: all SMs (the serial baseline and T_A alone on the GPU) and the budget the rule picks
        sms_list = sms_arg if sms_arg else [148, pipeline_attend_sms(Bm * S * 2 * Hkv * 128 * 2, weight_bytes_layer)]
        rec["attend_sms_rule"] = None if sms_arg else sms_list[1]
        for sms in sms_list:
            wls = [Workload(f"mb{m}_b{Bm}_s{S}", Hq, Hkv, R, P, [S] * Bm, seed=260629207 + m) for m in range(2)]
            total_steps = 40
            sess = [Session(wl, n_layers_phys=1, steps=total_steps, attend_sms=0 if sms >= 148 else sms) for wl in wls]
            for s_ in sess:
                s_.prepare()
            with torch.cuda.stream(ws):
                bufs = []
                for wl in wls:
                    bufs.append({"x": gen_device.fill_x(0, Bm, 0, hidden, seed=wl.seed),
                                 "q": torch.zeros((Bm, Hq, 128), dtype=torch.float16, device=dev),
                                 "k": torch.zeros((Bm, Hkv, 128), dtype=torch.float16, device=dev),
                                 "v": torch.zeros((Bm, Hkv, 128), dtype=torch.float16, device=dev),
                                 "o": torch.zeros((Bm, Hq, 128), dtype=torch.float32, device=dev),
                                 "lse": torch.zeros((Bm, Hq), dtype=torch.float32, device=dev)})
                x0 = [b["x"].clone() for b in bufs]
                layers = [l % Lw for l in range(n_layers)]
                b0 = bufs[0]
                if sms == sms_list[0]:
                    # stage times, each alone on the GPU
                    rec["T_p_us"] = graph_us(lambda i: (w.project_q(i % Lw, b0["x"], b0["q"], ws),
                                                        w.project_kv(i % Lw, b0["x"], b0["k"], b0["v"], ws)))
                    xs_ = torch.empty_like(b0["x"])
                    rec["T_f_us"] = graph_us(lambda i: w.post_attention(i % Lw, b0["o"], xs_, ws))
                kf0 = sess[0].kf
                kf0.token_boundary(ws)
                t_a = graph_us(lambda i: kf0.layer_step(0, b0["q"], b0["k"], b0["v"], b0["o"], b0["lse"], stream=ws))
                ws.synchronize()

                def step_us(mode):
                    """One decode step (n_layers layers x 2 microbatches) as ONE CUDA graph, replayed."""
                    w.set_sms(148 - sms if mode and sms < 148 else 0)      # the GEMMs get the SMs the attend grid leaves
                    def run():
                        w.pipeline_step([s_.kf for s_ in sess], layers, [b_["x"] for b_ in bufs], [b_["q"] for b_ in bufs],
                                        [b_["k"] for b_ in bufs], [b_["v"] for b_ in bufs], [b_["o"] for b_ in bufs],
                                        [b_["lse"] for b_ in bufs], mode, ws, as_)
                    run()
                    ws.synchronize()
                    g = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(g, stream=ws):
                        run()
                    ts = []
                    for i in range(8):
                        # x is overwritten in place by every layer and there is no norm between the layers: start every
                        # replay from the seeded hidden state, or fp16 would saturate after a few replays
                        for b_, x_ in zip(bufs, x0):
                            b_["x"].copy_(x_)
                        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        a.record(ws)
                        g.replay()
                        b.record(ws)
                        if i >= 2:
                            ts.append((a, b))
                    torch.cuda.synchronize(dev)
                    del g
                    w.set_sms(0)
                    finite.append(all(bool(torch.isfinite(b_["x"]).all()) for b_ in bufs))
                    return statistics.median(x.elapsed_time(y) for x, y in ts) * 1e3
                finite = []
                ser = step_us(0)
                pip = step_us(1)
                for s_ in sess:
                    assert s_.kf.status() == 0
            for s_ in sess:
                s_.close()
            del sess, bufs
            gc.collect()
            torch.cuda.empty_cache()
            per = {"attend_sms": sms, "T_A_us": t_a, "serial_us_per_layer_mb": ser / (2 * n_layers),
                   "pipelined_us_per_layer_mb": pip / (2 * n_layers), "measured_ratio": ser / pip,
                   "x_finite_after_step": all(finite)}
            rec.setdefault("by_sms", []).append(per)
            if best is None or per["pipelined_us_per_layer_mb"] < best["pipelined_us_per_layer_mb"]:
                best = per
        t_a148 = rec["by_sms"][0]["T_A_us"]
        tp, tf = rec["T_p_us"], rec["T_f_us"]
        kv_bytes = Bm * S * 4096
        rec["T_A_us"] = t_a148
        rec["model_G_pipe"] = (tp + t_a148 + tf) / max(tp + tf, t_a148)
        rec["serial_us_per_layer_mb"] = rec["by_sms"][0]["serial_us_per_layer_mb"]
        rec["serial_vs_sum_of_stages"] = rec["serial_us_per_layer_mb"] / (tp + t_a148 + tf)
        rec["best"] = best
        rec["measured_ratio_best"] = rec["serial_us_per_layer_mb"] / best["pipelined_us_per_layer_mb"]
        # what ONE GPU allows: both stages are bound by the same HBM, so a filled pipeline cannot beat bytes / bandwidth
        rec["bytes_per_layer_mb"] = weight_bytes_layer + kv_bytes
        rec["one_gpu_hbm_floor_us"] = (weight_bytes_layer + kv_bytes) / (peak * 1e9) * 1e6
        rec["W_side_GBs"] = weight_bytes_layer / ((tp + tf) * 1e-6) / 1e9
        rec["pipelined_GBs"] = (weight_bytes_layer + kv_bytes) / (best["pipelined_us_per_layer_mb"] * 1e-6) / 1e9
        if want_parity:
            rec["parity"] = pipeline_parity(w, Bm, S, R, P, best["attend_sms"], ws, as_)
        rows.append(rec)
    w.close()
    return {"mode": "pipeline", "model": "Llama-3.1-8B shape (hidden 4096, 32/8 heads, ffn 14336), synthetic weights",
            "weight_bytes_per_layer": weight_bytes_layer, "peak_gbs": peak, "peak_source": peak_src, "cases": rows}


_W_HOST = {}


def pipeline_parity(w, Bm, S, R, P, sms, ws, as_):
    """PARITY of the timed pipeline configuration, after its timing: fresh sessions (so the KV context is the generator's,
    not what the timed replays appended), the seeded hidden state, ONE pipelined kf_pipeline_step through layer 0 with the
    SM split that was timed -- and x' of two requests per microbatch against the oracle chain project -> append ->
    attend -> W_O -> SwiGLU FFN on the same inputs (tolerance: DESIGN.md section 6, the x' gate)."""
    import numpy as np
    import torch
    import oracle
    from oracle import wside as ow
    from kf_inputs import gen_device
    from kf_inputs.workloads import Workload
    from paper_2606_29207_b200 import KF_W_DOWN, KF_W_GATE, KF_W_KV, KF_W_O, KF_W_Q, KF_W_UP
    from paper_2606_29207_b200.workload import Session
    hidden, Hq, Hkv = 4096, 32, 8
    if "W" not in _W_HOST:
        _W_HOST["W"] = {k: w.weight(0, k).cpu().numpy() for k in (KF_W_Q, KF_W_KV, KF_W_O, KF_W_GATE, KF_W_UP, KF_W_DOWN)}
    W = _W_HOST["W"]
    wls = [Workload(f"mb{m}_b{Bm}_s{S}", Hq, Hkv, R, P, [S] * Bm, seed=260629207 + m) for m in range(2)]
    sess = [Session(wl, n_layers_phys=1, steps=2, attend_sms=0 if sms >= 148 else sms) for wl in wls]
    for s_ in sess:
        s_.prepare()
    dev = sess[0].device
    with torch.cuda.stream(ws):
        xs = [gen_device.fill_x(0, Bm, 0, hidden, seed=wl.seed) for wl in wls]
        x0 = [x.cpu().numpy() for x in xs]
        bufs = [{"q": torch.zeros((Bm, Hq, 128), dtype=torch.float16, device=dev),
                 "k": torch.zeros((Bm, Hkv, 128), dtype=torch.float16, device=dev),
                 "v": torch.zeros((Bm, Hkv, 128), dtype=torch.float16, device=dev),
                 "o": torch.zeros((Bm, Hq, 128), dtype=torch.float32, device=dev),
                 "lse": torch.zeros((Bm, Hq), dtype=torch.float32, device=dev)} for _ in wls]
        w.set_sms(148 - sms if sms < 148 else 0)
        ws.synchronize()
        w.pipeline_step([s_.kf for s_ in sess], [0], xs, [b["q"] for b in bufs], [b["k"] for b in bufs],
                        [b["v"] for b in bufs], [b["o"] for b in bufs], [b["lse"] for b in bufs], 1, ws, as_)
        ws.synchronize()
        as_.synchronize()
        w.set_sms(0)
        got = [x.cpu().numpy().astype(np.float64) for x in xs]
        ok_state = all(s_.kf.status() == 0 for s_ in sess)
    rows = [0, Bm - 1]
    xin = np.concatenate([x0[m][rows] for m in range(2)])                       # [4][hidden]
    pr = ow.project(xin, W[KF_W_Q], W[KF_W_KV])
    o = np.zeros((len(xin), Hq * 128))
    for i in range(len(xin)):
        m, r = divmod(i, len(rows))
        K, V = _host_kv(wls[m], rows[r], S - 1, True)
        K = np.concatenate([K, pr["k16"][i].reshape(Hkv, 1, 128)], 1)
        V = np.concatenate([V, pr["v16"][i].reshape(Hkv, 1, 128)], 1)
        o[i] = oracle.attend(pr["q16"][i].reshape(Hq, 128), np.ascontiguousarray(K), np.ascontiguousarray(V))[0].reshape(-1)
    ref = ow.post_attention(o, W[KF_W_O], W[KF_W_GATE], W[KF_W_UP], W[KF_W_DOWN])["x"]
    g = np.concatenate([got[m][rows] for m in range(2)])
    rms = float(np.sqrt(np.mean(ref * ref)))
    ratio = float((np.abs(g - ref) / (np.abs(ref) + rms + 1e-12)).max())
    finite = bool(all(np.isfinite(x).all() for x in got))
    for s_ in sess:
        s_.close()
    # the chain gate.  Unlike x' from an exact o (5 u), this chain carries the attend kernel's own
    # P-rounding noise (1..3 u of rms(o)) through W_O and the SwiGLU doubling: 4.4..6 u measured, gate 20 u
    gate = 1e-2
    return {"ok": bool(finite and ok_state and ratio <= gate), "max_err_over_ref_plus_rms": ratio, "gate": gate,
            "rows": len(xin), "x_finite": finite, "attend_sms": sms, "gemm_ctas": 148 - sms if sms < 148 else 148,
            "what": "one pipelined kf_pipeline_step (layer 0) from the seeded x, rows 0 and B-1 of both microbatches, vs "
                    "oracle project -> append -> attend -> W_O -> SwiGLU FFN"}


def compact_pipeline(full):
    """The `pipeline` record of the default line: one entry per case, numbers only."""
    out = []
    for c in full["cases"]:
        b = c["best"]
        out.append(_round({"B_mu": c["B_mu"], "seq": c["seq"], "T_p_us": c["T_p_us"], "T_f_us": c["T_f_us"], "T_A_us": c["T_A_us"],
                           "serial_us": c["serial_us_per_layer_mb"], "pipelined_us": b["pipelined_us_per_layer_mb"],
                           "attend_sms": b["attend_sms"], "attend_sms_rule": c.get("attend_sms_rule"),
                           "measured_ratio": c["measured_ratio_best"],
                           "model_G_pipe": c["model_G_pipe"], "one_gpu_hbm_floor_us": c["one_gpu_hbm_floor_us"],
                           "pipelined_over_floor": b["pipelined_us_per_layer_mb"] / c["one_gpu_hbm_floor_us"],
                           "x_finite": b["x_finite_after_step"],
                           "parity": {k: c["parity"][k] for k in ("ok", "max_err_over_ref_plus_rms", "gate", "rows")}
                           if c.get("parity") else None}))
    return {"layers_per_step": full["cases"][0]["layers_per_step"] if full["cases"] else None, "microbatches": 2,
            "unit": "us per (layer, microbatch)", "cases": out}


def run_pipeline(args):
    """--pipeline: the full table (every case x every SM budget of --pipe-sms, or the rule's budget with --pipe-sms rule)."""
    cases = [tuple(int(v) for v in c.split("x")) for c in args.pipe_cases.split(",")]
    sms_list = None if args.pipe_sms == "rule" else [int(v) for v in args.pipe_sms.split(",")]
    print(json.dumps(pipeline_cases(cases, sms_list, args.pipe_layers)))
    return 0




def run_wside_once(args):
    """--wside-once: every W-side stage once per batch size (after one untimed round), eagerly, on the 8B layer shape.
    Exists to be run under `ncu -k regex:wgemm`: the captures of wgemm_kernel / wgemm_fixup_kernel under profiles/."""
    import torch
    from kf_inputs import gen_device
    from paper_2606_29207_b200.workload import make_wside
    hidden, Hq, Hkv, ffn = 4096, 32, 8, 14336
    w = make_wside(hidden, Hq, Hkv, ffn, n_layers=1, max_batch=128)
    torch.cuda.synchronize()
    n0 = w.launch_count()
    for batch in (16, 128):
        x = gen_device.fill_x(0, batch, 0, hidden)
        q = torch.empty((batch, Hq, 128), dtype=torch.float16, device="cuda")
        k = torch.empty((batch, Hkv, 128), dtype=torch.float16, device="cuda")
        v = torch.empty_like(k)
        o = torch.randn((batch, Hq, 128), dtype=torch.float32, device="cuda")
        xn = torch.empty((batch, hidden), dtype=torch.float16, device="cuda")
        for _ in range(2):
            w.project_q(0, x, q)
            w.project_kv(0, x, k, v)
            w.post_attention(0, o, xn)
            torch.cuda.synchronize()
    print(json.dumps({"mode": "wside-once", "launches": w.launch_count() - n0}))
    w.close()
    return 0


def run_sm_sweep(args):
    """--sm-sweep: kf_attend GB/s against the SM budget of its persistent grid (kf_config.attend_sms)."""
    import statistics
    import torch
    from kf_inputs import workloads
    from paper_2606_29207_b200.workload import Session
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    wl = workloads.by_name(args.workload)
    out = {"mode": "sm-sweep", "workload": wl.name, "points": []}
    for sms in [int(v) for v in args.pipe_sms.split(",")]:
        ses = Session(wl, n_layers_phys=1, steps=4, attend_sms=0 if sms >= 148 else sms)
        ses.prepare()
        kf = ses.kf
        kf.token_boundary()
        q = ses.q_for(0, 0)
        k_new, v_new = ses.kv_new_for(0, 0)
        kf.kv_append(0, k_new, v_new)
        ts = []
        for i in range(25):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            kf.attend(0, q, ses.o, ses.lse)
            b.record()
            if i >= 5:
                ts.append((a, b))
        torch.cuda.synchronize()
        t = statistics.median(x.elapsed_time(y) for x, y in ts)
        nbytes = algorithmic_bytes(wl, list(ses.len0), 1)[0]
        out["points"].append({"attend_sms": sms, "attend_us": t * 1e3, "gbs": nbytes / (t * 1e-3) / 1e9})
        assert kf.status() == 0
        ses.close()
        del ses
        gc.collect()
        torch.cuda.empty_cache()
    print(json.dumps(out))
    return 0


# ---------------------------------------------------------------------------------------------------------
def measure_static(ses, wl, dev, reps=60, warm=5):
    """SURVEY 8(d) protocol for the static configs: the state is prepared once (S-1 tokens loaded, token boundary,
    append at position S-1) and `kf_kv_append + kf_attend` is repeated WITHOUT a commit, so every repetition attends
    over exactly the stated contexts.  Repetitions are replays of one captured graph of the two calls (the C-ABI calls
    are capturable); CUDA events around every replay; 512 MiB are written between replays when the KV fits L2."""
    import torch
    kf = ses.kf
    kf.token_boundary()
    q = ses.q_for(0, 0)
    k_new, v_new = ses.kv_new_for(0, 0)
    kf.layer_step(0, q, k_new, v_new, ses.o, ses.lse)
    torch.cuda.synchronize(dev)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=torch.cuda.current_stream(dev)):
        kf.layer_step(0, q, k_new, v_new, ses.o, ses.lse)      # a2 + a3 + a4 in one launch, as the step graph runs it
    lens = list(ses.len0)
    nbytes, kv = algorithmic_bytes(wl, lens, 1)
    flush = kv <= 4 * 126e6
    flush_buf = torch.empty(512 << 20, dtype=torch.uint8, device=dev) if flush else None
    ev = []
    for i in range(warm + reps):
        if flush:
            flush_buf.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        g.replay()
        b.record()
        if i >= warm:
            ev.append((a, b))
    torch.cuda.synchronize(dev)
    ts = sorted(a.elapsed_time(b) for a, b in ev)
    # the same launch eagerly, events around the call
    at = []
    for i in range(warm + 20):
        if flush:
            flush_buf.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        kf.layer_step(0, q, k_new, v_new, ses.o, ses.lse)
        b.record()
        if i >= warm:
            at.append((a, b))
    torch.cuda.synchronize(dev)
    att = sorted(a.elapsed_time(b) for a, b in at)
    assert kf.status() == 0
    del g, flush_buf
    med = ts[len(ts) // 2]
    # N repetitions inside ONE graph, replayed back to back: takes the ~2 us granularity of a CUDA event pair around a
    # single short launch out of the number
    n_in = 20
    g2 = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g2, stream=torch.cuda.current_stream(dev)):
        for _ in range(n_in):
            kf.layer_step(0, q, k_new, v_new, ses.o, ses.lse)
    b2b = []
    for i in range(8):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        g2.replay()
        b.record()
        if i >= 2:
            b2b.append((a, b))
    torch.cuda.synchronize(dev)
    b2b_us = sorted(a.elapsed_time(b) * 1e3 / n_in for a, b in b2b)
    assert kf.status() == 0
    del g2
    return {"protocol": "SURVEY 8(d) static: no commit between repetitions; kf_layer_step (append + attend + merge, one "
                        "launch) replayed as a graph",
            "back_to_back_us": b2b_us[len(b2b_us) // 2],
            "back_to_back_note": f"{n_in} repetitions in one graph, replayed back to back; L2-"
                                 + ("WARM (the KV fits L2)" if flush else "cold (KV >> L2)"),
            "context_tokens": sum(lens) + wl.batch, "algorithmic_bytes": nbytes,
            "us_per_layer_step_median": med * 1e3, "us_per_layer_step_min": ts[0] * 1e3,
            "value": nbytes / (med * 1e-3) / 1e9, "pct_of_nominal_8TBs": 100.0 * nbytes / (med * 1e-3) / 1e9 / NOMINAL_PEAK_GBS,
            "attend_us_median": att[len(att) // 2] * 1e3, "attend_us_min": att[0] * 1e3, "l2_flushed": bool(flush),
            "repetitions": reps}


def measure(args, wl_name, steps, warmup, e2e_steps, dev, dist, rank, world, local, want_cpu, want_probe=True,
            cpu_budget_s=15.0):
    """Everything bench.py reports for ONE workload; returns the record (rank 0) or None."""
    import torch
    from kf_inputs import workloads
    from paper_2606_29207_b200 import sharding
    from paper_2606_29207_b200.workload import Session

    t_wall0 = time.perf_counter()
    wl = workloads.by_name(wl_name)
    wl.seed = sharding.rank_seed(wl.seed, rank)    # independent batch per rank (weak scaling)
    n_layers = wl.n_layers
    total_steps = warmup + steps + 200 + e2e_steps + 4   # + the roofline and L2-warm regions (<= 100 steps each)
    if args.layers_phys:
        L_phys = args.layers_phys
    else:
        free, _ = torch.cuda.mem_get_info(dev)
        per_layer = wl.slots_per_partition(total_steps) * wl.n_partitions * wl.range_tokens * wl.kv_bytes_per_token()
        L_phys = max(1, min(n_layers, int(0.85 * free // per_layer)))
    ses = Session(wl, impl=args.attend_impl, n_layers_phys=L_phys, steps=total_steps, min_tiles=args.min_tiles,
                  device=str(dev), kv_l2_policy=args.kv_l2_policy, workers_per_sm=args.workers_per_sm,
                  pipeline_stages=args.stages)
    kf = ses.kf
    ses.prepare()
    assert kf.status() == 0
    prepare_s = time.perf_counter() - t_wall0

    static = None
    if n_layers == 1 and rank == 0 and not args.no_static:
        static = measure_static(ses, wl, dev)      # leaves len untouched (no commit): the loop below starts at step 0

    # per-step inputs, resident in HBM before the timed region (keyed by physical layer)
    def inputs(step):
        return [(ses.q_for(lp, step),) + ses.kv_new_for(lp, step) for lp in range(L_phys)]

    lens = list(ses.len0)

    def run_step(step_inputs, ev=None):
        kf.token_boundary()
        for layer in range(n_layers):
            q, kn, vn = step_inputs[layer % L_phys]
            if ev is not None:
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                kf.layer_step(layer % L_phys, q, kn, vn, ses.o, ses.lse)      # ONE launch: a2 + a3 + a4
                b.record()
                ev.append((a, b))
            else:
                kf.layer_step(layer % L_phys, q, kn, vn, ses.o, ses.lse)
        kf.step_commit()

    n_eager = max(1, warmup - 2)
    step = 0
    for _ in range(n_eager):
        run_step(inputs(step))
        step += 1
    assert kf.status() == 0

    # ---- the timed region: K decode steps, each ONE replay of the static step graph (kf_step_graph_*) with the
    #      step's resident inputs re-bound; --no-graph times the same calls launched one by one ---------------------
    layer_ids = [layer % L_phys for layer in range(n_layers)]

    def per_layer(step_inputs):
        return ([step_inputs[lp][0] for lp in layer_ids], [step_inputs[lp][1] for lp in layer_ids],
                [step_inputs[lp][2] for lp in layer_ids])

    o_list, lse_list = [ses.o] * n_layers, [ses.lse] * n_layers
    graph = None
    if not args.no_graph:
        q0, k0, v0 = per_layer(inputs(step))
        graph = kf.step_graph_create(layer_ids, q0, k0, v0, o_list, lse_list)

    def timed_step(step_inputs):
        if graph is None:
            run_step(step_inputs)
        else:
            q, kn, vn = per_layer(step_inputs)
            graph.launch(q, kn, vn, o_list, lse_list)

    for _ in range(warmup - n_eager):          # the last warm-up steps run exactly what is timed
        timed_step(inputs(step))
        step += 1
    resident = n_layers * steps <= 4096
    timed_inputs = [inputs(step + i) for i in range(steps)] if resident else None
    total_bytes = kv_bytes = 0
    for i in range(steps):
        b, k = algorithmic_bytes(wl, [n + step + i for n in lens], n_layers)
        total_bytes += b
        kv_bytes += k

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.15)
    torch.cuda.synchronize(dev)
    if dist:
        dist.barrier()
    launches0 = kf.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    # KV of one layer-step that fits L2 (cfg1: 16 MiB vs 126 MB) would be served from L2 after the first step:
    # write a 512 MiB buffer between timed steps, outside the per-step event windows, so `value` is an HBM number
    flush = kv_bytes / (steps * n_layers) <= 4 * 126e6 and not args.no_l2_flush
    flush_buf = torch.empty(512 << 20, dtype=torch.uint8, device=dev) if flush else None
    step_events = []
    t0 = sampler.mark()
    e0.record()
    for i in range(steps):
        if flush:
            flush_buf.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
        timed_step(timed_inputs[i] if timed_inputs else inputs(step + i))
        if flush:
            b.record()
            step_events.append((a, b))
    e1.record()
    torch.cuda.synchronize(dev)
    t1 = sampler.mark()
    if dist:
        dist.barrier()
    launches = kf.launch_count() - launches0
    step += steps
    ms = sum(a.elapsed_time(b) for a, b in step_events) if flush else e0.elapsed_time(e1)
    warm_ms_per_step = None
    if flush:        # the L2-warm number, reported beside it: the same steps back to back
        n_warm = min(steps, 100)
        warm_inputs = [inputs(step + i) for i in range(n_warm)]
        torch.cuda.synchronize(dev)
        e0.record()
        for i in range(n_warm):
            timed_step(warm_inputs[i])
        e1.record()
        torch.cuda.synchronize(dev)
        warm_ms_per_step = e0.elapsed_time(e1) / n_warm
        step += n_warm
    del timed_inputs
    assert kf.status() == 0

    # ---- roofline region: the same steps launched one by one, CUDA events around every kf_attend (events cannot
    #      be recorded inside a graph replay); also gives the eager step time ---------------------------------------
    roof_steps = max(1, min(steps, 4096 // n_layers, 100))
    roof_inputs = [inputs(step + i) for i in range(roof_steps)]
    attend_events = []
    r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(dev)
    r0.record()
    for i in range(roof_steps):
        if flush:
            flush_buf.zero_()
        run_step(roof_inputs[i], attend_events)
    r1.record()
    torch.cuda.synchronize(dev)
    eager_ms_per_step = None if flush else r0.elapsed_time(r1) / roof_steps   # (the flush writes sit in this region)
    attend_times = sorted(a.elapsed_time(b) for a, b in attend_events)
    attend_ms = sum(attend_times) / len(attend_times)
    roof_bytes = sum(algorithmic_bytes(wl, [n + step + i for n in lens], n_layers)[0] for i in range(roof_steps))
    attend_bytes = roof_bytes / (roof_steps * n_layers)  # per kf_attend launch (append rows are ~1e-5 of it)
    step += roof_steps
    del roof_inputs
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    assert kf.status() == 0

    # ---- read-only bandwidth probe over the same KV pools (third denominator; MEASURED_PEAKS' figure is a copy) ----
    probe_gbs = None
    pool_bytes = sum(p.numel() for p in kf.pools)
    if rank == 0 and want_probe and pool_bytes > 8 * 126e6:
        sink = torch.zeros(1, dtype=torch.int32, device=dev)
        best = None
        for _ in range(4):
            p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            p0.record()
            pool_bytes = kf.probe_read(sink)
            p1.record()
            torch.cuda.synchronize(dev)
            t = p0.elapsed_time(p1)
            best = t if best is None else min(best, t)
        probe_gbs = pool_bytes / (best * 1e-3) / 1e9
    ms, total_bytes_all, launches_all = sharding.aggregate(ms, total_bytes, launches, dist, dev)
    value = sharding.throughput_gbs(total_bytes_all, ms)
    ms_per_step = ms / steps

    # ---- end to end: HOST buffers, transfers inside the timed region.  One replay per step of a host-io step graph
    #      (pinned buffers): every layer-step reads q / k_new / v_new from host memory over the bus and
    #      writes o / lse to host memory; the caller reads the result on the host every step ---------------------------
    B, Hq, Hkv = wl.batch, wl.n_q_heads, wl.n_kv_heads
    host_in = []
    for i in range(e2e_steps):
        host_in.append([tuple(t.cpu().pin_memory() for t in x) for x in inputs(step + i)])
    qh = [torch.zeros((B, Hq, 128), dtype=torch.float16).pin_memory() for _ in range(n_layers)]
    kh = [torch.zeros((B, Hkv, 128), dtype=torch.float16).pin_memory() for _ in range(n_layers)]
    vh = [torch.zeros((B, Hkv, 128), dtype=torch.float16).pin_memory() for _ in range(n_layers)]
    o_h = [torch.zeros((B, Hq, 128), dtype=torch.float32).pin_memory() for _ in range(n_layers)]
    l_h = [torch.zeros((B, Hq), dtype=torch.float32).pin_memory() for _ in range(n_layers)]
    hgraph = None if args.no_graph else kf.step_graph_create(layer_ids, qh, kh, vh, o_h, l_h, host_io=True)
    e2e_bytes = 0
    for i in range(e2e_steps):
        e2e_bytes += algorithmic_bytes(wl, [n + step + i for n in lens], n_layers)[0]
    checksum = 0.0
    torch.cuda.synchronize(dev)
    if dist:
        dist.barrier()
    e0.record()
    for i in range(e2e_steps):
        if hgraph is None:
            kf.token_boundary()
            for layer in range(n_layers):
                qx, kx, vx = host_in[i][layer % L_phys]
                kf.layer_step_host(layer % L_phys, qx, kx, vx, o_h[layer], l_h[layer])
            kf.step_commit()
        else:                                       # this step's own pinned input buffers are re-bound
            hgraph.launch([host_in[i][lp][0] for lp in layer_ids], [host_in[i][lp][1] for lp in layer_ids],
                          [host_in[i][lp][2] for lp in layer_ids], o_h, l_h)
        torch.cuda.current_stream(dev).synchronize()      # the caller reads the step's result on the host
        checksum += float(l_h[n_layers - 1][0, 0])
    e1.record()
    torch.cuda.synchronize(dev)
    e2e_ms = e0.elapsed_time(e1)
    e2e_ms, e2e_bytes_all, _ = sharding.aggregate(e2e_ms, e2e_bytes, 0, dist, dev)
    step += e2e_steps
    e2e_value = sharding.throughput_gbs(e2e_bytes_all, e2e_ms)
    h2d = n_layers * (B * Hq * 128 * 2 + 2 * B * Hkv * 128 * 2)
    d2h = n_layers * (B * Hq * 128 * 4 + B * Hq * 4)
    assert kf.status() == 0 and checksum == checksum
    if hgraph is not None:
        hgraph.destroy()

    cpu = parity = None
    if rank == 0 and world == 1 and want_cpu:
        # ---- the oracle on the host cores (a baseline, not the target), and PARITY of this very step: one more decode
        #      step through the timed path (the static step graph), its (o, lse) compared with what the oracle just computed
        import numpy as np
        import oracle
        lens_now = [n + step for n in lens]
        chosen, data, desc = oracle_sample(wl, lens_now, cpu_budget_s, True)
        timed_step(inputs(step))                    # physical layer of the last layer-step: layer_ids[-1]
        torch.cuda.synchronize(dev)
        assert kf.status() == 0
        o_gpu, lse_gpu = ses.o.cpu().numpy().astype(np.float64), ses.lse.cpu().numpy().astype(np.float64)
        dt, ref = oracle_run(wl, chosen, data, step)
        nbytes = sum(n for _, n in chosen) * wl.kv_bytes_per_token()
        cpu = {"value": nbytes / dt / 1e9, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"{desc}, decode step {step}, {dt:.2f} s", "seconds": dt,
               "sample_short": f"{len(chosen)} of {B} requests, {sum(n for _, n in chosen)} context tokens"
                               + ("" if all(n == lens_now[r] + 1 for r, n in chosen) else " (prefix)")}
        if wl.name == "cfg1":       # SURVEY 8(d) "CPU baseline": the smallest config also on ONE thread
            dt1, _ = oracle_run(wl, chosen, data, step, n_threads=1)
            cpu["one_thread"] = {"value": nbytes / dt1 / 1e9, "seconds": dt1, "cores": 1}
        if layer_ids[-1] == 0 and all(n == lens_now[r] + 1 for r, n in chosen):
            eo = max(float(np.abs(o_gpu[r] - ref[r][0]).max()) for r, _ in chosen)
            el = max(float((np.abs(lse_gpu[r] - ref[r][1]) / np.maximum(1.0, np.abs(ref[r][1]))).max())
                     for r, _ in chosen)
            mo = max(float(np.abs(ref[r][0]).max()) for r, _ in chosen)
            parity = {"max_abs_o": eo, "max_rel_lse": el, "rows": len(chosen) * Hq, "requests": len(chosen),
                      "max_abs_o_ref": mo, "tol_abs_o": 2e-3, "tol_rel_lse": 1e-4,
                      "ok": bool(eo <= 2e-3 and el <= 1e-4),
                      "what": f"kf_step_graph replay of decode step {step} (all {Hq} heads of the sampled requests) vs "
                              "oracle.attend fp64 on the same inputs"}
        step += 1
        del data

    if graph is not None:
        graph.destroy()
    ses.close()
    del ses, kf, flush_buf
    gc.collect()
    torch.cuda.empty_cache()
    if rank != 0:
        return None

    peak, peak_src = load_peak()
    achieved = attend_bytes / (attend_ms * 1e-3) / 1e9
    traffic, traffic_src = traffic_record(wl.name, args)
    return {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f16 storage, f32 accumulate", "data": "synthetic",
        "config": {"workload": wl.name, "note": wl.note, "batch": B, "n_q_heads": Hq, "n_kv_heads": Hkv,
                   "range_tokens": wl.range_tokens, "n_partitions": wl.n_partitions, "layers_logical": n_layers,
                   "layers_physical": L_phys, "context_tokens_step0": sum(lens) + B,
                   "l2": "inputs larger than L2 (KV per layer-step >> 126 MB), no flush" if not flush and
                         kv_bytes / (steps * n_layers) > 4 * 126e6 else
                         "KV fits L2: 512 MiB written between timed steps outside the event windows (value is L2-cold, "
                         "warm_ms_per_step is back to back)" if flush else "KV fits L2, --no-l2-flush: L2-warm",
                   "attend_impl": {0: "tma", 1: "simple", 2: "tma"}[args.attend_impl],
                   "launch": "eager" if args.no_graph else "kf_step_graph replay per step, inputs re-bound",
                   "roofline_region": f"{roof_steps} further steps, CUDA events around every kf_layer_step launch"},
        "eager_ms_per_step": eager_ms_per_step, "warm_ms_per_step": warm_ms_per_step,
        "us_per_layer_step": ms_per_step * 1e3 / n_layers,
        "pct_of_nominal_8TBs": 100.0 * value / world / NOMINAL_PEAK_GBS,
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps},
        "gpu_launches": launches_all,
        "roofline": {"bound": "hbm", "kernel": "attend_tma_kernel" if args.attend_impl != 1 else "attend_simple_kernel",
                     "achieved": achieved, "peak": peak, "unit": UNIT, "frac": achieved / peak,
                     "traffic": traffic, "traffic_source": traffic_src.split(" (")[0], "kernel_rev": kernel_rev(),
                     "algorithmic_bytes_per_launch": int(round(attend_bytes)),
                     "avg_launch_ms": attend_ms, "median_launch_ms": attend_times[len(attend_times) // 2],
                     "min_launch_ms": attend_times[0], "launches_timed": len(attend_times), "peak_source": peak_src,
                     "frac_of_nominal_8000": achieved / NOMINAL_PEAK_GBS,
                     "read_probe_gbs": probe_gbs, "frac_of_read_probe": achieved / probe_gbs if probe_gbs else None},
        "static": static,
        "cpu_baseline": cpu,
        "parity": parity,
        "wall_s": {"prepare": prepare_s, "total": time.perf_counter() - t_wall0},
    }


# ---------------------------------------------------------------------------------------------------------
FIG10_DEFAULT = ["fig10_q32kv32_b32_s32k", "fig10_q48kv8_b32_s32k", "fig10_q64kv8_b32_s32k",
                 "fig10_q32kv32_b8_s8k", "fig10_q48kv8_b8_s8k", "fig10_q64kv8_b8_s8k"]
PIPELINE_DEFAULT = [(16, 2048), (64, 8192), (128, 4096)]


def run_extras(args, dev, local):
    """The records of the default line beyond BASELINE's five configs, each compact: `fig10` (head shapes G = 1 / 6 / 8 at
    two sizes: PAPER.md:322), `signalling` (route install, token boundary, flag round trip: PAPER.md:308, :165-175) and
    `pipeline` (three of Fig. 11's workloads: PAPER.md:335-337) -- so that one driver-run line carries every number the
    profiles quote."""
    import torch
    out = {}
    t0 = time.perf_counter()
    fig = {}
    for name in FIG10_DEFAULT:
        rec = measure(args, name, 30, 5, 10, dev, None, 0, 1, local, want_cpu=False, want_probe=False)
        fig[name] = _round({"us_per_layer_step": rec["us_per_layer_step"], "value": rec["value"],
                            "frac": rec["roofline"]["frac"], "frac_of_nominal_8000": rec["roofline"]["frac_of_nominal_8000"],
                            "static_us": rec["static"]["us_per_layer_step_median"] if rec.get("static") else None,
                            "e2e": rec["e2e"]["value"]})
    out["fig10"] = fig
    t1 = time.perf_counter()
    out["signalling"] = _round(signalling_record(torch.device(f"cuda:{local}")))
    t2 = time.perf_counter()
    cur = torch.cuda.current_stream(dev)
    out["pipeline"] = compact_pipeline(pipeline_cases(PIPELINE_DEFAULT, None, 8))
    torch.cuda.set_stream(cur)
    out["extras_wall_s"] = _round({"fig10": t1 - t0, "signalling": t2 - t1, "pipeline": time.perf_counter() - t2}, 3)
    return out


def wl_steps_note(line):
    return f"all {line['config']['n_q_heads']} query heads, layer 0, oracle.attend fp64"


def _round(x, sig=5):
    """Floats to `sig` significant digits, recursively: the JSON line stays short enough for a log tail."""
    if isinstance(x, float):
        return float(f"{x:.{sig}g}") if x == x and abs(x) != float("inf") else x
    if isinstance(x, dict):
        return {k: _round(v, sig) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_round(v, sig) for v in x]
    return x


def compact_record(rec):
    """The sub-record of one workload inside the headline line: numbers only, no prose (the full record of a workload
    is what `bench.py --workload <name> --only` prints)."""
    ro, st, cpu, par = rec["roofline"], rec.get("static"), rec.get("cpu_baseline"), rec.get("parity")
    out = {"value": rec["value"], "us_per_layer_step": rec["us_per_layer_step"],
           "pct_of_nominal_8TBs": rec["pct_of_nominal_8TBs"], "steps": rec["steps"], "warmup": rec["warmup"],
           "warm_ms_per_step": rec.get("warm_ms_per_step"), "gpu_launches": rec["gpu_launches"],
           "e2e": {"value": rec["e2e"]["value"], "ms_per_step": rec["e2e"]["ms_per_step"]},
           "roofline": {"achieved": ro["achieved"], "frac": ro["frac"], "traffic": ro["traffic"],
                        "avg_launch_ms": ro["avg_launch_ms"], "algorithmic_bytes_per_launch": int(ro["algorithmic_bytes_per_launch"]),
                        "frac_of_read_probe": ro["frac_of_read_probe"]},       # peak: the headline's roofline.peak
           "clocks": {"sm_mhz": rec["clocks"].get("sm_mhz"), "reasons": rec["clocks"].get("reasons")},
           "config": {k: rec["config"][k] for k in ("batch", "n_q_heads", "n_kv_heads", "layers_logical",
                                                    "layers_physical", "context_tokens_step0")}}
    if st:
        out["static"] = {k: st[k] for k in ("us_per_layer_step_median", "back_to_back_us", "attend_us_median", "value",
                                            "pct_of_nominal_8TBs", "l2_flushed")}
    if cpu:
        out["cpu_baseline"] = {k: cpu[k] for k in ("value", "cores", "seconds", "one_thread") if k in cpu}
        out["cpu_baseline"]["sample"] = cpu["sample_short"]
    if par:
        out["parity"] = {k: par[k] for k in ("ok", "max_abs_o", "max_rel_lse", "rows")}
    r = _round(out)
    r["roofline"]["traffic"], r["roofline"]["algorithmic_bytes_per_launch"] = out["roofline"]["traffic"], out["roofline"]["algorithmic_bytes_per_launch"]
    return r


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--workload", default="cfg3", help="the headline workload of the JSON line")
    ap.add_argument("--only", action="store_true", help="measure the headline workload only (no `workloads` sub-records)")
    ap.add_argument("--sub", default=",".join(SUB_WORKLOADS), help="comma-separated sub-record workloads")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--attend-impl", type=int, default=0, help="KF_IMPL_*: 0 auto, 1 simple, 2 tma")
    ap.add_argument("--layers-phys", type=int, default=0, help="physical layer pools (0 = auto)")
    ap.add_argument("--e2e-steps", type=int, default=0, help="0 = min(steps, 50)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--min-tiles", type=int, default=0)
    ap.add_argument("--workers-per-sm", type=int, default=0, help="kf_config.workers_per_sm (0 = default)")
    ap.add_argument("--stages", type=int, default=0, help="kf_config.pipeline_stages (0 = default)")
    ap.add_argument("--kv-l2-policy", type=int, default=0, help="kf_config.kv_l2_policy: 0 default, 1 evict-first, 2 normal")
    ap.add_argument("--route-install", action="store_true", help="measure the latency of a scale event (route "
                    "install) and of the token boundary instead of the decode benchmark")
    ap.add_argument("--no-l2-flush", action="store_true", help="do not flush L2 between timed steps when the KV of a "
                    "layer-step fits L2 (cfg1)")
    ap.add_argument("--no-graph", action="store_true", help="launch the calls of a step one by one instead of "
                    "replaying the static step graph")
    ap.add_argument("--no-static", action="store_true", help="skip the static (no-commit) protocol")
    ap.add_argument("--pipeline", action="store_true", help="measure the W-side stages and the M = 2 inter-layer pipeline "
                    "(PAPER.md:252-280) instead of the decode benchmark")
    ap.add_argument("--pipe-cases", default="16x2048,16x8192,16x16384,32x4096,64x2048,64x8192,128x2048,128x4096,128x16384",
                    help="--pipeline workloads: B_mu x seq (Fig. 11: batch 16-128, sequence 2K-16K)")
    ap.add_argument("--pipe-sms", default="148,116,100,84,68", help="attend SM budgets tried by --pipeline / --sm-sweep")
    ap.add_argument("--pipe-layers", type=int, default=8, help="layers per step in --pipeline")
    ap.add_argument("--sm-sweep", action="store_true", help="kf_attend GB/s against its SM budget")
    ap.add_argument("--wside-once", action="store_true", help="run every W-side stage once per batch size (for ncu captures)")
    ap.add_argument("--no-extras", action="store_true", help="skip the `fig10`, `signalling` and `pipeline` records of the "
                    "default line")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.route_install:
        return run_route_install(args)
    if args.pipeline:
        return run_pipeline(args)
    if args.sm_sweep:
        return run_sm_sweep(args)
    if args.wside_once:
        return run_wside_once(args)
    args.warmup = max(args.warmup, 3)

    import torch

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device(f"cuda:{local}")
    torch.cuda.set_stream(torch.cuda.Stream(dev))   # stream capture (kf_step_graph_create) needs a non-default stream
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    e2e_steps = args.e2e_steps or min(args.steps, 50)
    line = measure(args, args.workload, args.steps, args.warmup, e2e_steps, dev, dist, rank, world, local,
                   want_cpu=not args.no_cpu_baseline)
    subs = {}
    if not args.only and world == 1:
        for name in [w for w in args.sub.split(",") if w and w != args.workload]:
            st, wu, e2 = SUB_STEPS.get(name, (50, 5, 20))
            # the oracle is timed per config as well (SURVEY 8(d) "CPU baseline"), on a ~3 s sample each
            rec = measure(args, name, st, wu, e2, dev, None, 0, 1, local, want_cpu=not args.no_cpu_baseline,
                          want_probe=name != "cfg1", cpu_budget_s=3.0)
            subs[name] = compact_record(rec)
    extras = {}
    if not args.only and world == 1 and not args.no_extras:
        extras = run_extras(args, dev, local)
    if rank == 0:
        if subs:
            line["workloads"] = subs
        line.update(extras)
        if not args.only:      # the all-in-one line is kept short (numbers to 6 digits, prose cut): it has to survive a log tail
            exact = {k: line[k] for k in ("value", "ms_per_step")}
            if line.get("static"):
                line["static"] = {k: v for k, v in line["static"].items() if k not in ("protocol", "back_to_back_note")}
            if line.get("cpu_baseline"):
                line["cpu_baseline"]["sample"] = line["cpu_baseline"].pop("sample_short") + f", {wl_steps_note(line)}"
            if line.get("parity"):
                line["parity"].pop("what", None)
            line["config"].pop("note", None)
            line = _round(line, 6)
            line.update(exact)
        print(json.dumps(line))
    if dist:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
