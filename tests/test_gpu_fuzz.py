"""Seeded random decode loops through the C ABI against the fp64 oracle and the integer routing model: random head
shapes (G = 1..8), range sizes (1..256 tokens), partition counts, batch sizes, context lengths, chunk granularity,
plan refresh periods, fused / unfused paths.  Small sizes, many shapes: aimed at edge cases of the work plan
(scheduling levels of tiny units, kept plans crossing tile and range edges, ragged tiles)."""
import random

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from kf_inputs.workloads import Workload  # noqa: E402
from kf_testlib import check_close, oracle_request  # noqa: E402
from oracle.routing import RoutingModel  # noqa: E402
from paper_2606_29207_b200 import KF_IMPL_SIMPLE, KF_IMPL_TMA, KF_OK  # noqa: E402
from paper_2606_29207_b200.workload import Session  # noqa: E402


def _one_case(rnd, case):
    Hkv = rnd.choice([1, 2, 4, 8])
    G = rnd.choice([1, 2, 3, 4, 6, 8])
    R = rnd.choice([1, 4, 16, 32, 64, 256])
    P = rnd.randrange(1, 6)
    B = rnd.randrange(1, 10)
    hi = rnd.choice([8, 40, 300, 900])
    ctx = [rnd.randrange(1, min(hi, 40 * R) + 1) for _ in range(B)]
    steps = rnd.randrange(1, 6)
    impl = KF_IMPL_SIMPLE if case % 7 == 6 else KF_IMPL_TMA
    fused = rnd.random() < 0.7
    one_launch = fused and rnd.random() < 0.5      # kf_layer_step: append + attend + merge in one launch
    wl = Workload(f"fuzz{case}", Hkv * G, Hkv, R, P, ctx)
    ses = Session(wl, impl=impl, steps=steps, min_tiles=rnd.choice([0, 0, 1, 2]),
                  plan_refresh_steps=rnd.choice([0, 0, 1, 2]), sched_decay_pct=rnd.choice([0, 30, 70]))
    ses.prepare()
    kf = ses.kf
    model = RoutingModel(P, R, B, kf.Jmax, kf.cfg.slots_per_partition)
    for r, n in enumerate(ses.len0):
        model.open_request(r, n)
    what = f"case {case}: Hkv={Hkv} G={G} R={R} P={P} ctx={ctx} steps={steps} impl={impl} fused={fused} one_launch={one_launch}"
    for t in range(steps):
        kf.token_boundary()
        model.token_boundary()
        q = ses.q_for(0, t)
        k_new, v_new = ses.kv_new_for(0, t)
        ses.o.fill_(float("nan"))
        ses.lse.fill_(float("nan"))
        ses.layer_step(0, q, k_new, v_new, fused=fused, one_launch=one_launch)
        kf.step_commit()
        model.step_commit()
        assert kf.status() == KF_OK, what
        o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
        assert np.isfinite(o).all() and np.isfinite(lse).all(), what
        for r in rnd.sample(range(B), min(B, 3)):
            o_ref, lse_ref = oracle_request(wl, 0, r, t, ctx[r] + t)
            check_close(o[r], lse[r], o_ref, lse_ref, f"{what} step {t} r{r}")
    snap, ms = kf.route_snapshot(), model.snapshot()
    for key in ("len", "n_ranges", "part", "slot", "free_head", "rr_cursor"):
        assert snap[key] == ms[key], f"{what}: {key}"
    ses.close()


@pytest.mark.parametrize("block", range(4))
def test_random_decode_loops(block):
    rnd = random.Random(1000 + block)
    for i in range(10):
        _one_case(rnd, 10 * block + i)


@pytest.mark.parametrize("G", [5, 7])
@pytest.mark.parametrize("impl", [KF_IMPL_SIMPLE, KF_IMPL_TMA])
def test_odd_group_sizes(impl, G):
    # kf_config admits every G = H_q / H_kv in 1..8; the random draws above only reach {1, 2, 3, 4, 6, 8}.  G = 5 and 7
    # leave the last rows of the kernel's 8-row query tile empty and make the merge tasks' head chunks ragged.
    # Ragged contexts over several ranges and partitions, three decode steps, fused / unfused / one launch; routes vs the
    # integer model, every request and every range partial vs the oracle (which maps h -> h / G itself).
    Hkv = 2
    wl = Workload(f"odd_g{G}", Hkv * G, Hkv, 32, 3, [1, 17, 32, 33, 100, 257], n_steps=3)
    ses = Session(wl, impl=impl, steps=3)
    ses.prepare()
    kf = ses.kf
    model = RoutingModel(3, 32, wl.batch, kf.Jmax, kf.cfg.slots_per_partition)
    for r, n in enumerate(ses.len0):
        model.open_request(r, n)
    for step in range(3):
        kf.token_boundary()
        model.token_boundary()
        q = ses.q_for(0, step)
        k_new, v_new = ses.kv_new_for(0, step)
        ses.layer_step(0, q, k_new, v_new, fused=step != 1, want_partials=True,
                       one_launch=step == 2 and impl == KF_IMPL_TMA)
        kf.step_commit()
        model.step_commit()
        assert kf.status() == KF_OK
        o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
        op, lp = ses.o_part.cpu().numpy(), ses.lse_part.cpu().numpy()
        for r, S0 in enumerate(wl.contexts):
            o_ref, lse_ref, op_ref, lp_ref = oracle_request(wl, 0, r, step, S0 + step, ranges=True)
            check_close(o[r], lse[r], o_ref, lse_ref, f"G{G} step{step} r{r}")
            J = op_ref.shape[0]
            check_close(op[r, :J], lp[r, :J], op_ref, lp_ref, f"G{G} step{step} r{r} partials")
    snap, ms = kf.route_snapshot(), model.snapshot()
    for key in ("len", "n_ranges", "part", "slot", "free_head", "rr_cursor"):
        assert snap[key] == ms[key], key
    ses.close()
