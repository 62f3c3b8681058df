"""GPU tests of kf_step_graph_*: one decode step as a static CUDA graph, replayed across range fills, route
updates and open/close of requests with no re-capture (the single-GPU analogue of PAPER.md:127 R1, :165-179)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from kf_inputs import gen, gen_device  # noqa: E402
from kf_inputs.workloads import Workload  # noqa: E402
from kf_testlib import check_close, oracle_request  # noqa: E402
from oracle.routing import RoutingModel  # noqa: E402
from paper_2606_29207_b200 import KF_EINVAL, KF_OK, KFlumeError  # noqa: E402
from paper_2606_29207_b200.workload import Session  # noqa: E402


def _check_step(ses, wl, layer, step, o, lse, what):
    for r, S0 in enumerate(wl.contexts):
        o_ref, lse_ref = oracle_request(wl, layer, r, step, S0 + step)
        check_close(o[r], lse[r], o_ref, lse_ref, f"{what} layer{layer} step{step} r{r}")


def test_step_graph_replay_across_route_updates_with_rebinding():
    # two physical layers; request 1 fills its 64-token range at step 3, request 3 at step 0 (opens at the first
    # boundary); inputs of every step live in their own tensors, so every launch re-binds q / k_new / v_new
    wl = Workload("graph", 32, 8, 64, 3, [200, 125, 33, 65, 16], n_layers=2)
    steps = 24
    ses = Session(wl, steps=steps)
    ses.prepare()
    kf = ses.kf
    model = RoutingModel(wl.n_partitions, wl.range_tokens, wl.batch, kf.Jmax, kf.cfg.slots_per_partition)
    for r, n in enumerate(ses.len0):
        model.open_request(r, n)
    B, Hq = wl.batch, wl.n_q_heads
    o = [torch.zeros((B, Hq, 128), dtype=torch.float32, device="cuda") for _ in range(2)]
    lse = [torch.zeros((B, Hq), dtype=torch.float32, device="cuda") for _ in range(2)]
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        ins = [[(ses.q_for(l, t),) + ses.kv_new_for(l, t) for l in range(2)] for t in range(steps)]
        g = kf.step_graph_create([0, 1], [ins[0][l][0] for l in range(2)], [ins[0][l][1] for l in range(2)],
                                 [ins[0][l][2] for l in range(2)], o, lse)
        launches0 = kf.launch_count()
        for t in range(steps):
            q = [ins[t][l][0] for l in range(2)]
            kn = [ins[t][l][1] for l in range(2)]
            vn = [ins[t][l][2] for l in range(2)]
            g.launch(q, kn, vn, o, lse)
            model.token_boundary()
            model.step_commit()
            side.synchronize()
            for l in range(2):
                _check_step(ses, wl, l, t, o[l].cpu().numpy(), lse[l].cpu().numpy(), "graph")
        # plan, 2 x attend: the append of each layer-step and the commit of the step ride in the attend launches
        assert kf.launch_count() - launches0 == steps * 3
        assert kf.status() == KF_OK
        snap, ms = kf.route_snapshot(), model.snapshot()
        for key in ("len", "n_ranges", "part", "slot", "free_head", "rr_cursor"):
            assert snap[key] == ms[key], key
        assert sum(ms["n_ranges"]) > sum(-(-n // 64) for n in ses.len0)     # ranges were opened during replay
        # (a2) rides in the attend launch of the graph: every appended row of every step / layer / request / kv head
        # sits bit-exact where the integer model puts it
        for l in range(2):
            for r, n0 in enumerate(ses.len0):
                K = gen_device.fill(gen.STREAM_K, l, r, n0, steps, wl.n_kv_heads, seed=wl.seed)
                V = gen_device.fill(gen.STREAM_V, l, r, n0, steps, wl.n_kv_heads, seed=wl.seed)
                for t in range(steps):
                    p, sl, off = model.locate(r, n0 + t)
                    for gk in range(wl.n_kv_heads):
                        for is_v, src in ((False, K), (True, V)):
                            o0 = kf.pool_offset(l, sl, gk, off, is_v)
                            assert torch.equal(kf.pools[p][o0:o0 + 256].view(torch.float16), src[gk, t]), (l, r, t, gk, is_v)
        g.destroy()
    ses.close()


def test_step_graph_matches_eager_bit_for_bit_and_survives_close_open():
    wl = Workload("graph_eq", 32, 8, 128, 2, [300, 45, 129, 127])
    steps = 12

    def run(use_graph):
        ses = Session(wl, steps=steps, slack_slots=2)
        ses.prepare()
        kf = ses.kf
        side = torch.cuda.Stream()
        outs = []
        with torch.cuda.stream(side):
            q, (kn, vn) = ses.q_for(0, 0), ses.kv_new_for(0, 0)
            qs, ks, vs = q.clone(), kn.clone(), vn.clone()      # static input buffers, rewritten every step
            g = kf.step_graph_create([0], [qs], [ks], [vs], [ses.o], [ses.lse]) if use_graph else None
            for t in range(steps):
                if t == 5:          # host-side route edit between replays: request 1 leaves, its slot is reused
                    kf.close_request(1)
                    kf.open_request(1, 44 + t)
                    k, v = ses_kv(ses, wl, 1, 44 + t)
                    kf.load_context(0, 1, 0, k, v)
                q, (kn, vn) = ses.q_for(0, t), ses.kv_new_for(0, t)
                qs.copy_(q), ks.copy_(kn), vs.copy_(vn)
                if use_graph:
                    g.launch()
                else:
                    kf.token_boundary()
                    ses.layer_step(0, qs, ks, vs)
                    kf.step_commit()
                side.synchronize()
                outs.append((ses.o.cpu().numpy().copy(), ses.lse.cpu().numpy().copy()))
            assert kf.status() == KF_OK
            if g is not None:
                g.destroy()
        ses.close()
        return outs

    a, b = run(True), run(False)
    for t, ((oa, la), (ob, lb)) in enumerate(zip(a, b)):
        assert np.array_equal(oa, ob) and np.array_equal(la, lb), t
    for t in (0, 4, 5, 11):
        for r, S0 in enumerate(wl.contexts):
            o_ref, lse_ref = oracle_request(wl, 0, r, t, S0 + t)
            check_close(a[t][0][r], a[t][1][r], o_ref, lse_ref, f"graph_eq step{t} r{r}")


def ses_kv(ses, wl, req, n):
    from kf_inputs import gen, gen_device
    k = gen_device.fill(gen.STREAM_K, 0, req, 0, n, wl.n_kv_heads, seed=wl.seed)
    v = gen_device.fill(gen.STREAM_V, 0, req, 0, n, wl.n_kv_heads, seed=wl.seed)
    return k, v


def test_step_graph_host_io_matches_device_path():
    wl = Workload("graph_host", 32, 8, 128, 2, [300, 45, 129])
    steps = 6
    ses = Session(wl, steps=steps)
    ses.prepare()
    kf = ses.kf
    B, Hq, Hkv = wl.batch, wl.n_q_heads, wl.n_kv_heads
    qh = torch.zeros((B, Hq, 128), dtype=torch.float16).pin_memory()
    kh = torch.zeros((B, Hkv, 128), dtype=torch.float16).pin_memory()
    vh = torch.zeros((B, Hkv, 128), dtype=torch.float16).pin_memory()
    oh = torch.zeros((B, Hq, 128), dtype=torch.float32).pin_memory()
    lh = torch.zeros((B, Hq), dtype=torch.float32).pin_memory()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        g = kf.step_graph_create([0], [qh], [kh], [vh], [oh], [lh], host_io=True)
        pageable = torch.zeros((B, Hq, 128), dtype=torch.float16)
        with pytest.raises(KFlumeError) as ei:       # host pointers must be pinned: the kernels read them directly
            g.launch([pageable], [kh], [vh], [oh], [lh])
        assert ei.value.code == KF_EINVAL
        oh2, lh2 = torch.zeros_like(oh).pin_memory(), torch.zeros_like(lh).pin_memory()
        for t in range(steps):
            q, (kn, vn) = ses.q_for(0, t), ses.kv_new_for(0, t)
            side.synchronize()
            if t % 2 == 0:           # rewrite the bound buffers ...
                qh.copy_(q.cpu()), kh.copy_(kn.cpu()), vh.copy_(vn.cpu())
                g.launch([qh], [kh], [vh], [oh], [lh])
                out = (oh, lh)
            else:                    # ... or re-bind to this step's own pinned buffers
                g.launch([q.cpu().pin_memory()], [kn.cpu().pin_memory()], [vn.cpu().pin_memory()], [oh2], [lh2])
                out = (oh2, lh2)
            side.synchronize()
            _check_step(ses, wl, 0, t, out[0].numpy(), out[1].numpy(), "graph_host")
        assert kf.status() == KF_OK
        g.destroy()
    ses.close()
