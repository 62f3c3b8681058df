"""GPU tests of graph progress signalling (kf_step_graph_flags): WriteValue32-style readiness
flags written by the static step graph into host-visible memory, ReadValue32-style gates released by a host thread on
a dedicated signalling stream, the same-stream hazard of PAPER.md:175, and results that still match the fp64 oracle
while scale events edit the routing table between replays -- all without re-capturing the graph."""
import ctypes
import threading
import time

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from kf_inputs.workloads import Workload  # noqa: E402
from kf_testlib import check_close, oracle_request  # noqa: E402
from oracle.routing import RoutingModel  # noqa: E402
from paper_2606_29207_b200 import KF_EINVAL, KF_ESTATE, KF_OK, KFlumeError  # noqa: E402
from paper_2606_29207_b200.workload import Session  # noqa: E402


def _spin_until(arr, i, value, timeout_s=20.0):
    t0 = time.perf_counter()
    while int(arr[i]) != value:
        if time.perf_counter() - t0 > timeout_s:
            return False
    return True


def test_host_thread_feeds_and_drains_a_running_graph_in_order():
    # two layer-steps per decode step, pinned host buffers; the "CPU routing loop" (a host thread) writes the inputs of
    # layer-step i, releases gate i on the signalling stream, waits for readiness flag i and takes the outputs -- while
    # the ONE graph launch of that step is still in flight.  Scale events between replays; nothing is re-captured.
    wl = Workload("flags", 32, 8, 32, 4, [70, 31, 33, 100, 64], n_layers=2)
    steps, n = 30, 2
    ses = Session(wl, steps=steps, slack_slots=8)
    kf = ses.kf
    model = RoutingModel(4, 32, wl.batch, kf.Jmax, kf.cfg.slots_per_partition)
    active = [1, 1, 0, 0]
    kf.set_active_partitions(active)
    model.set_active(active)
    ses.prepare()
    for r, m in enumerate(ses.len0):
        model.open_request(r, m)
    B, Hq, Hkv = wl.batch, wl.n_q_heads, wl.n_kv_heads
    qh = [torch.zeros((B, Hq, 128), dtype=torch.float16).pin_memory() for _ in range(n)]
    kh = [torch.zeros((B, Hkv, 128), dtype=torch.float16).pin_memory() for _ in range(n)]
    vh = [torch.zeros((B, Hkv, 128), dtype=torch.float16).pin_memory() for _ in range(n)]
    oh = [torch.full((B, Hq, 128), float("nan"), dtype=torch.float32).pin_memory() for _ in range(n)]
    lh = [torch.full((B, Hq), float("nan"), dtype=torch.float32).pin_memory() for _ in range(n)]
    ready = torch.zeros(n, dtype=torch.int32).pin_memory()
    ready_np = ready.numpy()
    events = {6: [1, 1, 1, 0], 12: [0, 1, 1, 0], 18: [0, 1, 1, 1]}
    side, signal = torch.cuda.Stream(), torch.cuda.Stream()
    observed, results, errors = [], {}, []
    with torch.cuda.stream(side):
        g = kf.step_graph_create([0, 1], qh, kh, vh, oh, lh, host_io=True)
        g.flags(ready, gates=True)
        ins = [[tuple(x.cpu() for x in ((ses.q_for(l, t),) + ses.kv_new_for(l, t))) for l in range(n)]
               for t in range(steps)]
        side.synchronize()

        def routing_loop(t, seqs):
            try:
                for i in range(n):
                    qh[i].copy_(ins[t][i][0]), kh[i].copy_(ins[t][i][1]), vh[i].copy_(ins[t][i][2])
                    g.release(i, seqs[i], signal)                    # dedicated signalling stream
                    if not _spin_until(ready_np, i, seqs[i]):
                        errors.append(f"step {t}: readiness flag {i} never reached {seqs[i]}")
                        return
                    observed.append((i, int(ready_np[i])))
                    results[(t, i)] = (oh[i].numpy().copy(), lh[i].numpy().copy())   # outputs are complete NOW
            except Exception as e:          # noqa: BLE001
                errors.append(repr(e))
            finally:                        # whatever happened: never leave the graph waiting at a gate
                for j in range(n):
                    try:
                        g.release(j, seqs[j], signal)
                    except Exception:       # noqa: BLE001
                        pass

        for t in range(steps):
            if t in events:
                kf.set_active_partitions(events[t])
                model.set_active(events[t])
            seqs = [g.seq(i) for i in range(n)]
            assert seqs == [t * n + i + 1 for i in range(n)]
            g.launch()                                   # blocks at gate 0 on the device; the host call returns
            th = threading.Thread(target=routing_loop, args=(t, seqs))
            th.start()
            th.join(60)
            assert not th.is_alive() and not errors, errors
            side.synchronize()
            model.token_boundary()
            model.step_commit()
        assert kf.status() == KF_OK
        g.destroy()
    # flags were seen in order, one per layer-step of every replay
    assert observed == [(i, t * n + i + 1) for t in range(steps) for i in range(n)]
    for t in range(steps):
        for i in range(n):
            o, lse = results[(t, i)]
            for r, S0 in enumerate(wl.contexts):
                o_ref, lse_ref = oracle_request(wl, i, r, t, S0 + t)
                check_close(o[r], lse[r], o_ref, lse_ref, f"flags step{t} layer{i} r{r}")
    snap, ms = kf.route_snapshot(), model.snapshot()
    for key in ("len", "n_ranges", "part", "slot", "free_head", "rr_cursor"):
        assert snap[key] == ms[key], key
    ses.close()


def test_gate_really_blocks_and_same_stream_release_is_refused():
    # the execution stream is blocked on the wait, a flag write enqueued on it would sit behind the wait
    wl = Workload("flags_gate", 32, 8, 64, 2, [200, 33, 65])
    ses = Session(wl, steps=4)
    ses.prepare()
    kf = ses.kf
    side, signal = torch.cuda.Stream(), torch.cuda.Stream()
    ready = torch.zeros(1, dtype=torch.int32).pin_memory()
    with torch.cuda.stream(side):
        q, (kn, vn) = ses.q_for(0, 0), ses.kv_new_for(0, 0)
        g = kf.step_graph_create([0], [q], [kn], [vn], [ses.o], [ses.lse])
        pageable = np.zeros(1, np.int32)                             # pageable memory is not host-visible to the GPU
        assert kf.lib.kf_step_graph_flags(g.h, ctypes.c_void_p(pageable.ctypes.data), 1, kf._stream()) == KF_EINVAL
        g.flags(ready, gates=True)
        side.synchronize()
        ses.o.fill_(float("nan"))
        side.synchronize()
        seq = g.seq(0)
        g.launch()
        time.sleep(0.05)
        assert not side.query()                                     # the graph is waiting at its gate
        assert int(ready[0]) == 0                                   # (nothing may be enqueued on `side` here)
        with pytest.raises(KFlumeError) as ei:
            g.release(0, seq, side)                                 # same stream: would deadlock -> refused
        assert ei.value.code == KF_ESTATE
        g.release(0, seq, signal)                                   # the fix: a dedicated signalling stream
        side.synchronize()
        assert int(ready[0]) == seq
        o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
        for r, S0 in enumerate(wl.contexts):
            o_ref, lse_ref = oracle_request(wl, 0, r, 0, S0)
            check_close(o[r], lse[r], o_ref, lse_ref, f"gate r{r}")
        # a gate may be released BEFORE the launch that waits on it: the replay then runs straight through
        seq = g.seq(0)
        g.release(0, seq, signal)
        signal.synchronize()
        q1, (k1, v1) = ses.q_for(0, 1), ses.kv_new_for(0, 1)
        g.launch([q1], [k1], [v1], [ses.o], [ses.lse])
        side.synchronize()
        assert int(ready[0]) == seq == 2
        o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
        for r, S0 in enumerate(wl.contexts):
            o_ref, lse_ref = oracle_request(wl, 0, r, 1, S0 + 1)
            check_close(o[r], lse[r], o_ref, lse_ref, f"gate step1 r{r}")
        with pytest.raises(KFlumeError) as ei:                      # flags cannot be changed once launched
            g.flags(ready, gates=False)
        assert ei.value.code == KF_ESTATE
        assert kf.status() == KF_OK
        g.destroy()
    ses.close()


def test_readiness_flags_without_gates_and_roundtrip_latency():
    wl = Workload("flags_ready", 32, 8, 64, 2, [100, 17], n_layers=3)
    ses = Session(wl, steps=3)
    ses.prepare()
    kf = ses.kf
    side, signal = torch.cuda.Stream(), torch.cuda.Stream()
    ready = torch.zeros(3, dtype=torch.int32).pin_memory()
    with torch.cuda.stream(side):
        ins = [(ses.q_for(l, 0),) + ses.kv_new_for(l, 0) for l in range(3)]
        o = [torch.zeros_like(ses.o) for _ in range(3)]
        lse = [torch.zeros_like(ses.lse) for _ in range(3)]
        g = kf.step_graph_create([0, 1, 2], [x[0] for x in ins], [x[1] for x in ins], [x[2] for x in ins], o, lse)
        g.flags(ready, gates=False)
        g.launch()
        side.synchronize()
        assert ready.tolist() == [1, 2, 3]
        for l in range(3):
            oh, lh = o[l].cpu().numpy(), lse[l].cpu().numpy()
            for r, S0 in enumerate(wl.contexts):
                o_ref, lse_ref = oracle_request(wl, l, r, 0, S0)
                check_close(oh[r], lh[r], o_ref, lse_ref, f"ready layer{l} r{r}")
        g.destroy()
        med, mn = kf.signal_roundtrip(200, side, signal)
        assert 0.5 < mn <= med < 2000.0, (med, mn)                  # microseconds
        assert kf.status() == KF_OK
    ses.close()


def test_release_right_after_flags_survives_while_the_capture_stream_is_busy():
    # kflume.h: "a gate may be released before the launch that waits on it".  kf_step_graph_flags zeroes the gate words
    # on `stream`; if that memset could still be queued behind earlier work when a release on the signalling stream
    # lands, it would erase the release and the launch below would wait for ever.  Keep `side` busy (a long device-side
    # spin), call flags(), release at once, and only then let the stream drain.
    wl = Workload("flags_early", 32, 8, 64, 2, [200, 33, 65])
    ses = Session(wl, steps=2)
    ses.prepare()
    kf = ses.kf
    side, signal = torch.cuda.Stream(), torch.cuda.Stream()
    ready = torch.zeros(1, dtype=torch.int32).pin_memory()
    with torch.cuda.stream(side):
        q, (kn, vn) = ses.q_for(0, 0), ses.kv_new_for(0, 0)
        g = kf.step_graph_create([0], [q], [kn], [vn], [ses.o], [ses.lse])
        side.synchronize()
        ses.o.fill_(float("nan"))
        torch.cuda._sleep(400_000_000)                              # ~0.2 s of queued work in front of flags()
        g.flags(ready, gates=True)                                  # no synchronize() here, on purpose
        seq = g.seq(0)
        g.release(0, seq, signal)                                   # early release, before the launch exists
        signal.synchronize()
        g.launch()
        t0 = time.perf_counter()
        while not side.query() and time.perf_counter() - t0 < 20.0:
            time.sleep(0.005)
        done = side.query()
        if not done:                                                # never leave the GPU waiting at a gate
            g.release(0, seq, signal)
            side.synchronize()
        assert done, "the early release was erased: the graph was still waiting at its gate after 20 s"
        assert int(ready[0]) == seq
        assert kf.status() == KF_OK
        o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
        for r, S0 in enumerate(wl.contexts):
            o_ref, lse_ref = oracle_request(wl, 0, r, 0, S0)
            check_close(o[r], lse[r], o_ref, lse_ref, f"early release r{r}")
        g.destroy()
    ses.close()


def test_route_install_latency_probe_restores_the_active_set():
    # kf_route_install_latency toggles the active set `iters` times from C and must leave the one it found
    wl = Workload("install_probe", 32, 8, 64, 5, [100, 17, 64])
    ses = Session(wl, steps=2)
    ses.prepare()
    kf = ses.kf
    kf.set_active_partitions([1, 0, 1, 1, 0])
    before = kf.partition_state()
    n0 = kf.launch_count()
    enq, done = kf.route_install_latency(300)
    assert 0.0 < enq <= done < 5000.0, (enq, done)
    assert kf.launch_count() - n0 >= 311
    after = kf.partition_state()
    assert after["active"] == before["active"] == [1, 0, 1, 1, 0]
    assert kf.status() == KF_OK
    # and decoding goes on as if nothing had happened
    kf.token_boundary()
    q = ses.q_for(0, 0)
    k_new, v_new = ses.kv_new_for(0, 0)
    ses.layer_step(0, q, k_new, v_new)
    kf.step_commit()
    assert kf.status() == KF_OK
    o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
    for r, S0 in enumerate(wl.contexts):
        o_ref, lse_ref = oracle_request(wl, 0, r, 0, S0)
        check_close(o[r], lse[r], o_ref, lse_ref, f"after the probe r{r}")
    ses.close()
