"""GPU tests of kf_redirect_tails (Algorithm 1 l.16-17 taken literally; reading 28):
at the next token boundary the tails on a marked node are closed where they are and continue in a new, variable-length
range on an active node.  Routes, slots, range begins and occupancy bit-exact against the integer model; appended rows
bit-exact where the model locates them; attention against the fp64 oracle; eager, one-launch and static-graph paths."""
import random

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from kf_inputs import gen, gen_device  # noqa: E402
from kf_inputs.workloads import Workload  # noqa: E402
from kf_testlib import check_close, oracle_request  # noqa: E402
from oracle.routing import RoutingModel  # noqa: E402
from paper_2606_29207_b200 import KF_IMPL_SIMPLE, KF_IMPL_TMA, KF_OK  # noqa: E402
from paper_2606_29207_b200.workload import Session  # noqa: E402

KEYS = ("len", "n_ranges", "part", "slot", "begin", "free_head", "rr_cursor")


def _same(kf, model, what=""):
    snap, ms = kf.route_snapshot(), model.snapshot()
    for key in KEYS:
        assert snap[key] == ms[key], (what, key)
    assert kf.partition_state() == model.partition_state(), what


def _check_rows(ses, wl, model, layer, steps):
    kf = ses.kf
    for r, n0 in enumerate(ses.len0):
        K = gen_device.fill(gen.STREAM_K, layer, r, 0, n0 + steps, wl.n_kv_heads, seed=wl.seed)
        V = gen_device.fill(gen.STREAM_V, layer, r, 0, n0 + steps, wl.n_kv_heads, seed=wl.seed)
        for pos in range(n0 + steps):          # loaded context AND appended tokens, wherever the cuts put them
            p, sl, off = model.locate(r, pos)
            for gk in range(wl.n_kv_heads):
                for is_v, src in ((False, K), (True, V)):
                    o0 = kf.pool_offset(layer, sl, gk, off, is_v)
                    assert torch.equal(kf.pools[p][o0:o0 + 256].view(torch.float16), src[gk, pos]), (r, pos, gk, is_v)


def test_fig5_with_a_cut_at_t_plus_k_on_device():
    # the hand-worked pin of tests/test_oracle_routing.py, on the device: T = 16, R = 8, three nodes
    wl = Workload("fig5cut", 8, 2, 8, 3, [17])               # 16 tokens resident before step 0
    ses = Session(wl, steps=16, slack_slots=3, slack_ranges=3)
    kf = ses.kf
    model = RoutingModel(3, 8, 1, kf.Jmax, kf.cfg.slots_per_partition)
    ses.prepare()
    model.open_request(0, 16)
    for t in range(12):
        if t == 3:                                           # len = 19: node A2 leaves the set, its tails are redirected
            kf.set_active_partitions([1, 1, 0])
            kf.redirect_tails([0, 0, 1])
            model.set_active([1, 1, 0])
            model.redirect_tails([0, 0, 1])
        kf.token_boundary()
        model.token_boundary()
        _same(kf, model, f"step {t}")
        q, (kn, vn) = ses.q_for(0, t), ses.kv_new_for(0, t)
        ses.layer_step(0, q, kn, vn, one_launch=t % 2 == 0)
        kf.step_commit()
        model.step_commit()
        assert kf.status() == KF_OK
        o_ref, lse_ref = oracle_request(wl, 0, 0, t, 17 + t)
        check_close(ses.o[0].cpu().numpy(), ses.lse[0].cpu().numpy(), o_ref, lse_ref, f"fig5cut step {t}")
    snap = kf.route_snapshot()
    assert snap["begin"][0][:5] == [0, 8, 16, 19, 27] and snap["part"][0][:5] == [0, 1, 2, 0, 1]
    _check_rows(ses, wl, model, 0, 12)
    ses.close()


@pytest.mark.parametrize("impl", [KF_IMPL_SIMPLE, KF_IMPL_TMA])
@pytest.mark.parametrize("seed", [1, 2])
def test_random_redirects_closed_loop(impl, seed):
    # several requests, ranges of 32 tokens on 4 nodes, random scale events and redirects over 40 steps; every step:
    # routing state == model, every request's attention == oracle (partials per variable-length range included)
    rnd = random.Random(100 * seed + impl)
    wl = Workload(f"redir{seed}", 32, 8, 32, 4, [70, 31, 33, 100, 64, 1])
    steps = 40
    ses = Session(wl, impl=impl, steps=steps, slack_slots=40, slack_ranges=40, min_tiles=rnd.choice([0, 1]))
    kf = ses.kf
    model = RoutingModel(4, 32, wl.batch, kf.Jmax, kf.cfg.slots_per_partition)
    ses.prepare()
    for r, n in enumerate(ses.len0):
        model.open_request(r, n)
    n_cut = 0
    for t in range(steps):
        if rnd.random() < 0.3:
            act = [rnd.random() < 0.7 for _ in range(4)]
            act = act if any(act) else [1, 1, 1, 1]
            kf.set_active_partitions(act)
            model.set_active(act)
            parts = [0 if a else 1 for a in act] if rnd.random() < 0.6 else [rnd.random() < 0.5 for _ in range(4)]
            kf.redirect_tails(parts)
            model.redirect_tails(parts)
        kf.token_boundary()
        ev = model.token_boundary()
        n_cut += sum(1 for (r, j, _, _) in ev if model.begin[r][j] - model.begin[r][j - 1] < 32) if ev else 0
        _same(kf, model, f"step {t}")
        q, (kn, vn) = ses.q_for(0, t), ses.kv_new_for(0, t)
        for x in (ses.o, ses.lse, ses.o_part, ses.lse_part):
            x.fill_(float("nan"))
        ses.layer_step(0, q, kn, vn, fused=t % 3 != 2, want_partials=True, one_launch=t % 3 == 0)
        kf.step_commit()
        model.step_commit()
        assert kf.status() == KF_OK
        o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
        op, lp = ses.o_part.cpu().numpy(), ses.lse_part.cpu().numpy()
        for r, S0 in enumerate(wl.contexts):
            o_ref, lse_ref = oracle_request(wl, 0, r, t, S0 + t)
            check_close(o[r], lse[r], o_ref, lse_ref, f"redir step {t} r{r}")
            # per-range partials over the variable-length ranges [begin_j, begin_j+1)
            b = model.begin[r] + [S0 + t]
            K = gen.gen_k(0, r, np.arange(S0 + t), 8, wl.seed)
            V = gen.gen_v(0, r, np.arange(S0 + t), 8, wl.seed)
            qh = gen.gen_q(0, r, t, 32, wl.seed)
            import oracle
            for j in range(len(b) - 1):
                oj, lj = oracle.attend(qh, K[:, b[j]:b[j + 1]], V[:, b[j]:b[j + 1]])
                check_close(op[r, j], lp[r, j], oj, lj, f"redir step {t} r{r} range {j}")
    assert n_cut >= 3                                          # tails really were cut mid-range
    _check_rows(ses, wl, model, 0, steps)
    ses.close()


def test_redirect_through_the_static_graph_and_context_reload():
    # the step graph is captured BEFORE any redirect; the cuts happen during replay; afterwards kf_load_context
    # rewrites a span that crosses two cuts (position -> variable-length range lookup)
    wl = Workload("redir_graph", 32, 8, 64, 3, [200, 125, 33, 65])
    steps = 24
    ses = Session(wl, steps=steps, slack_slots=12, slack_ranges=12)
    kf = ses.kf
    model = RoutingModel(3, 64, wl.batch, kf.Jmax, kf.cfg.slots_per_partition)
    ses.prepare()
    for r, n in enumerate(ses.len0):
        model.open_request(r, n)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        ins = [(ses.q_for(0, t),) + ses.kv_new_for(0, t) for t in range(steps)]
        g = kf.step_graph_create([0], [ins[0][0]], [ins[0][1]], [ins[0][2]], [ses.o], [ses.lse])
        for t in range(steps):
            if t in (4, 9, 15):
                marked = [t == 4, t == 9, t == 15]
                kf.set_active_partitions([0 if m else 1 for m in marked])
                kf.redirect_tails(marked)
                model.set_active([0 if m else 1 for m in marked])
                model.redirect_tails(marked)
            g.launch([ins[t][0]], [ins[t][1]], [ins[t][2]], [ses.o], [ses.lse])
            model.token_boundary()
            model.step_commit()
            side.synchronize()
            o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
            for r, S0 in enumerate(wl.contexts):
                o_ref, lse_ref = oracle_request(wl, 0, r, t, S0 + t)
                check_close(o[r], lse[r], o_ref, lse_ref, f"redir graph step {t} r{r}")
        assert kf.status() == KF_OK
        _same(kf, model, "after replay")
        assert any(b[j + 1] - b[j] < 64 for b in model.begin for j in range(len(b) - 1))
        _check_rows(ses, wl, model, 0, steps)
        # reload request 0 completely with OTHER bytes (the generator's layer-1 values) through kf_load_context
        n = ses.len0[0] + steps
        K1 = gen_device.fill(gen.STREAM_K, 1, 0, 0, n, wl.n_kv_heads, seed=wl.seed)
        V1 = gen_device.fill(gen.STREAM_V, 1, 0, 0, n, wl.n_kv_heads, seed=wl.seed)
        kf.load_context(0, 0, 0, K1, V1)
        side.synchronize()
        assert kf.status() == KF_OK
        for pos in range(n):
            p, sl, off = model.locate(0, pos)
            for gk in (0, wl.n_kv_heads - 1):
                o0 = kf.pool_offset(0, sl, gk, off, False)
                assert torch.equal(kf.pools[p][o0:o0 + 256].view(torch.float16), K1[gk, pos]), pos
        g.destroy()
    ses.close()
