"""GPU tests of scale events: kf_set_active_partitions publishes a new active set of (emulated) attention nodes at a
token boundary; future ranges go to the new node, existing ranges stay (Fig. 5 at :173).
Routes, slots and occupancy are compared bit-exact with the integer model; attention with the fp64 oracle."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from kf_inputs.workloads import Workload  # noqa: E402
from kf_testlib import check_close, oracle_request  # noqa: E402
from oracle.routing import RoutingModel  # noqa: E402
from paper_2606_29207_b200 import KF_EINVAL, KF_OK, KFlumeError  # noqa: E402
from paper_2606_29207_b200.workload import Session  # noqa: E402


def _same(kf, model):
    snap, ms = kf.route_snapshot(), model.snapshot()
    for key in ("len", "n_ranges", "part", "slot", "free_head", "rr_cursor"):
        assert snap[key] == ms[key], key
    assert kf.partition_state() == model.partition_state()


def test_fig5_scale_up_on_device():
    R = 8
    wl = Workload("fig5", 8, 2, R, 3, [2 * R + 1])           # len before step 0 = 2R = T
    ses = Session(wl, steps=4, slack_slots=2)
    kf = ses.kf
    model = RoutingModel(3, R, 1, kf.Jmax, kf.cfg.slots_per_partition)
    kf.set_active_partitions([1, 1, 0])
    model.set_active([1, 1, 0])
    ses.open_all()
    model.open_request(0, 2 * R)
    _same(kf, model)
    assert kf.route_snapshot()["part"][0][:2] == [0, 1]
    kf.set_active_partitions([1, 1, 1])                       # route install of the prewarmed node
    model.set_active([1, 1, 1])
    kf.token_boundary()
    model.token_boundary()
    _same(kf, model)
    snap = kf.route_snapshot()
    assert snap["part"][0][:3] == [0, 1, 2] and snap["slot"][0][:3] == [0, 0, 0]
    with pytest.raises(KFlumeError) as ei:
        kf.set_active_partitions([0, 0, 0])
    assert ei.value.code == KF_EINVAL
    ses.close()


def test_scale_up_and_down_during_graph_replay_matches_model_and_oracle():
    # 4 partitions, 2 active at first; node 2 joins at step 6, node 0 retires at step 12, node 3 joins at step 18.
    # Ranges of 32 tokens fill every few steps, so every event redirects real allocations.
    wl = Workload("elastic", 32, 8, 32, 4, [70, 31, 33, 100, 64])
    steps = 30
    ses = Session(wl, steps=steps, slack_slots=8)
    kf = ses.kf
    model = RoutingModel(4, 32, wl.batch, kf.Jmax, kf.cfg.slots_per_partition)
    active = [1, 1, 0, 0]
    kf.set_active_partitions(active)
    model.set_active(active)
    ses.prepare()
    for r, n in enumerate(ses.len0):
        model.open_request(r, n)
    _same(kf, model)
    events = {6: [1, 1, 1, 0], 12: [0, 1, 1, 0], 18: [0, 1, 1, 1]}
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        q, (kn, vn) = ses.q_for(0, 0), ses.kv_new_for(0, 0)
        qs, ks, vs = q.clone(), kn.clone(), vn.clone()
        g = kf.step_graph_create([0], [qs], [ks], [vs], [ses.o], [ses.lse])     # captured ONCE, before any event
        for t in range(steps):
            if t in events:
                kf.set_active_partitions(events[t])
                model.set_active(events[t])
            q, (kn, vn) = ses.q_for(0, t), ses.kv_new_for(0, t)
            qs.copy_(q), ks.copy_(kn), vs.copy_(vn)
            g.launch()
            opened = model.token_boundary()
            for (_, _, p, _) in opened:
                assert model.active[p]                       # new ranges only on active nodes
            model.step_commit()
            side.synchronize()
            o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
            for r, S0 in enumerate(wl.contexts):
                o_ref, lse_ref = oracle_request(wl, 0, r, t, S0 + t)
                check_close(o[r], lse[r], o_ref, lse_ref, f"elastic step{t} r{r}")
            if t in (5, 11, 17, steps - 1):
                _same(kf, model)
        assert kf.status() == KF_OK
        g.destroy()
    st = kf.partition_state()
    assert st["active"] == [0, 1, 1, 1] and st["tokens"][3] > 0 and sum(st["tails"]) == wl.batch
    ses.close()


# ---- Algorithm 1 closed loop: the library's controller drives the device routing table -----------------------------
def _controller_loop(steps, P, state_fn, decide_fn, publish_fn, step_fn, prewarm_steps=3, redirect_fn=None):
    """The per-step monitor of Algorithm 1 around an abstract backend.  A node that reaches its watermark with a ready
    prewarm leaves the active set and the lowest-numbered idle node joins it: "redirect active tails on i to
    prewarm[i]" (l.17) under the fixed-R reading -- the tails move as their current ranges fill.  The joining node is a
    FRESH one (never provisioned before), as in the paper; with none left the event is skipped."""
    active = [1] + [0] * (P - 1)
    fresh = list(range(1, P))                     # nodes never provisioned so far, in bring-up order
    pending, ready, countdown = [False] * P, [False] * P, [0] * P
    history = []
    publish_fn(active)
    for t in range(steps):
        st = state_fn()
        dec = decide_fn(st["tokens"], st["tails"], pending, ready)
        for i, (_, spawn, publish) in enumerate(dec):
            if not active[i]:
                continue          # already published away: it only drains its tails' current ranges (<= R tokens each)
            if spawn:
                pending[i], countdown[i] = True, prewarm_steps
            if publish and fresh:
                active[fresh.pop(0)] = 1
                active[i] = 0
                ready[i] = False
                publish_fn(active)
                if redirect_fn is not None:   # l.17 literally (reading 28): node i's tails move at the next boundary
                    redirect_fn([1 if p == i else 0 for p in range(P)])
        for i in range(P):
            if pending[i]:
                countdown[i] -= 1
                if countdown[i] == 0:
                    pending[i], ready[i] = False, True
        history.append((list(active), list(st["tokens"]), list(st["tails"])))
        step_fn(t)
    return history


def test_algorithm1_closed_loop_device_equals_model():
    from oracle import policy as opol
    from paper_2606_29207_b200 import Policy
    P, R, steps = 4, 32, 200
    wl = Workload("alg1", 32, 8, R, P, [70, 31, 33, 100, 64])
    kw = dict(beta_mem=1.0, beta_slo=1.0, gamma=0.8, t_a_max_s=1.0, bw_hbm=1e30, c_kv_cap=4096.0 * 400,
              t_step_s=1.0, t_prewarm_s=3.0, n_kv_heads=8, head_dim=128, n_layers=1)
    pol, oc = Policy(**kw), opol.PolicyConstants(**kw)
    assert pol.initial_nodes([s - 1 for s in wl.contexts]) == 1          # 298 tokens fit one 400-token node

    ses = Session(wl, steps=steps, slack_slots=16)
    kf = ses.kf
    kf.set_active_partitions([1, 0, 0, 0])
    ses.prepare()

    def gpu_step(t):
        kf.token_boundary()
        q, (kn, vn) = ses.q_for(0, t), ses.kv_new_for(0, t)
        ses.layer_step(0, q, kn, vn)
        kf.step_commit()
        if t % 9 == 0 or t == steps - 1:
            o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
            for r, S0 in enumerate(wl.contexts):
                o_ref, lse_ref = oracle_request(wl, 0, r, t, S0 + t)
                check_close(o[r], lse[r], o_ref, lse_ref, f"alg1 step{t} r{r}")

    h_gpu = _controller_loop(steps, P, kf.partition_state, pol.step, kf.set_active_partitions, gpu_step)

    model = RoutingModel(P, R, wl.batch, kf.Jmax, kf.cfg.slots_per_partition)
    model.set_active([1, 0, 0, 0])
    for r, n in enumerate(ses.len0):
        model.open_request(r, n)

    def model_step(t):
        model.token_boundary()
        model.step_commit()

    h_model = _controller_loop(steps, P, model.partition_state,
                               lambda tok, tails, pe, re: opol.monitor(oc, tok, tails, pe, re), model.set_active, model_step)
    assert h_gpu == h_model                                   # same decisions, same occupancy, every step
    _same(kf, model)
    assert kf.status() == KF_OK
    actives = [tuple(a) for a, _, _ in h_gpu]
    assert len(set(actives)) >= 3                             # the policy scaled at least twice
    final_tokens = h_gpu[-1][1]
    assert sum(1 for x in final_tokens if x > 0) >= 3
    # a node stops receiving ranges once published away; it may still grow until its tails' current ranges fill
    assert max(final_tokens[:3]) <= 400 + wl.batch * R        # (the last node has no successor to hand over to)
    ses.close()


def test_algorithm1_closed_loop_with_tail_redirect_stops_growth_at_once():
    # the same controller, acting on want_publish as Algorithm 1 l.16-17 says: publish the route AND redirect the active
    # tails of node i (kf_redirect_tails, reading 28).  Device == model every step, and a retired node holds exactly
    # what it held at the boundary after the publish -- no overshoot of up to (tails * R) tokens as under reading 20.
    from oracle import policy as opol
    from paper_2606_29207_b200 import Policy
    P, R, steps = 4, 32, 200
    wl = Workload("alg1r", 32, 8, R, P, [70, 31, 33, 100, 64])
    kw = dict(beta_mem=1.0, beta_slo=1.0, gamma=0.8, t_a_max_s=1.0, bw_hbm=1e30, c_kv_cap=4096.0 * 400,
              t_step_s=1.0, t_prewarm_s=3.0, n_kv_heads=8, head_dim=128, n_layers=1)
    pol, oc = Policy(**kw), opol.PolicyConstants(**kw)
    ses = Session(wl, steps=steps, slack_slots=16, slack_ranges=8)
    kf = ses.kf
    kf.set_active_partitions([1, 0, 0, 0])
    ses.prepare()

    def gpu_step(t):
        kf.token_boundary()
        q, (kn, vn) = ses.q_for(0, t), ses.kv_new_for(0, t)
        ses.layer_step(0, q, kn, vn, one_launch=True)
        kf.step_commit()
        if t % 9 == 0 or t == steps - 1:
            o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
            for r, S0 in enumerate(wl.contexts):
                o_ref, lse_ref = oracle_request(wl, 0, r, t, S0 + t)
                check_close(o[r], lse[r], o_ref, lse_ref, f"alg1r step{t} r{r}")

    h_gpu = _controller_loop(steps, P, kf.partition_state, pol.step, kf.set_active_partitions, gpu_step,
                             redirect_fn=kf.redirect_tails)
    model = RoutingModel(P, R, wl.batch, kf.Jmax, kf.cfg.slots_per_partition)
    model.set_active([1, 0, 0, 0])
    for r, n in enumerate(ses.len0):
        model.open_request(r, n)

    def model_step(t):
        model.token_boundary()
        model.step_commit()

    h_model = _controller_loop(steps, P, model.partition_state,
                               lambda tok, tails, pe, re: opol.monitor(oc, tok, tails, pe, re), model.set_active,
                               model_step, redirect_fn=model.redirect_tails)
    assert h_gpu == h_model
    snap, ms = kf.route_snapshot(), model.snapshot()
    for key in ("len", "n_ranges", "part", "slot", "begin", "free_head", "rr_cursor"):
        assert snap[key] == ms[key], key
    assert kf.status() == KF_OK
    n_events = 0
    for t in range(1, steps - 1):
        a0, a1 = h_gpu[t - 1][0], h_gpu[t][0]
        for i in range(P):
            if a0[i] and not a1[i]:                       # node i was published away during iteration t - 1 ...
                n_events += 1
                assert h_gpu[t][2][i] > 0 or h_gpu[t][1][i] > 0
                assert h_gpu[t + 1][2][i] == 0            # ... one boundary later it holds no tail any more
                assert all(h[1][i] == h_gpu[t + 1][1][i] for h in h_gpu[t + 1:])   # and never grows again
    assert n_events >= 2
    ses.close()


def test_paused_requests_sit_out_steps():
    # requests pause and resume between decode steps (kf_set_active_requests); paused rows are untouched, their
    # length and routes frozen; everything else matches the oracle and the model at every step
    wl = Workload("pause", 32, 8, 32, 3, [70, 32, 33, 100, 64, 5])
    steps = 14
    ses = Session(wl, steps=steps, slack_slots=4)
    ses.prepare()
    kf = ses.kf
    B = wl.batch
    model = RoutingModel(3, 32, B, kf.Jmax, kf.cfg.slots_per_partition)
    for r, n in enumerate(ses.len0):
        model.open_request(r, n)
    schedule = {0: [1, 0, 1, 1, 0, 1], 4: [1, 1, 0, 1, 0, 1], 8: [0, 1, 1, 0, 1, 1], 11: None}
    act = [1] * B
    lens = list(ses.len0)
    pos_dev = torch.tensor(lens, dtype=torch.int32, device="cuda")
    from kf_inputs import gen, gen_device
    for t in range(steps):
        if t in schedule:
            mask = schedule[t]
            act = [1] * B if mask is None else mask
            kf.set_active_requests(None if mask is None else torch.tensor(mask, dtype=torch.uint8, device="cuda"))
            model.set_active_requests(mask)
        kf.token_boundary()
        model.token_boundary()
        q = ses.q_for(0, t)
        # K/V_new of a request is the generator value at ITS OWN next position (paused requests do not advance)
        pos_dev.copy_(torch.tensor(lens, dtype=torch.int32))
        k_new = gen_device.fill_rows(gen.STREAM_K, 0, pos_dev, wl.n_kv_heads, seed=wl.seed)
        v_new = gen_device.fill_rows(gen.STREAM_V, 0, pos_dev, wl.n_kv_heads, seed=wl.seed)
        ses.o.fill_(float("nan"))
        ses.lse.fill_(float("nan"))
        ses.layer_step(0, q, k_new, v_new)
        kf.step_commit()
        model.step_commit()
        assert kf.status() == KF_OK
        o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
        for r in range(B):
            if act[r]:
                o_ref, lse_ref = oracle_request(wl, 0, r, t, lens[r] + 1)
                check_close(o[r], lse[r], o_ref, lse_ref, f"pause step{t} r{r}")
                lens[r] += 1
            else:
                assert np.isnan(o[r]).all() and np.isnan(lse[r]).all(), (t, r)
        _same(kf, model)
        assert kf.route_snapshot()["len"] == lens
    ses.close()
