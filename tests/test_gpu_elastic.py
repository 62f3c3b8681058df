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
