"""GPU parity of the decode LOOP when the device work plan is kept across steps:
between rebuilds only the tail range of every request grows, and the attend kernels re-derive its extent from
`len` at run time.  Every step is checked against the fp64 oracle; routes against the integer model."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from kf_inputs.workloads import Workload  # noqa: E402
from kf_testlib import check_close, oracle_request  # noqa: E402
from oracle.routing import RoutingModel  # noqa: E402
from paper_2606_29207_b200 import KF_ESTATE, KF_IMPL_SIMPLE, KF_IMPL_TMA, KF_OK  # noqa: E402
from paper_2606_29207_b200.workload import Session  # noqa: E402

IMPLS = [KF_IMPL_SIMPLE, KF_IMPL_TMA]


def _decode_loop(wl, impl, steps, refresh, fused=True, min_tiles=0, check_every=1, one_launch=False):
    ses = Session(wl, impl=impl, steps=steps, min_tiles=min_tiles, plan_refresh_steps=refresh)
    ses.prepare()
    kf = ses.kf
    model = RoutingModel(wl.n_partitions, wl.range_tokens, wl.batch, kf.Jmax, kf.cfg.slots_per_partition)
    for r, n in enumerate(ses.len0):
        model.open_request(r, n)
    outs = []
    for step in range(steps):
        kf.token_boundary()
        model.token_boundary()
        q = ses.q_for(0, step)
        k_new, v_new = ses.kv_new_for(0, step)
        ses.o.fill_(float("nan"))
        ses.lse.fill_(float("nan"))
        ses.layer_step(0, q, k_new, v_new, fused=fused, one_launch=one_launch)
        kf.step_commit()
        model.step_commit()
        assert kf.status() == KF_OK
        o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
        outs.append((o.copy(), lse.copy()))
        if step % check_every == 0 or step == steps - 1:
            for r, S0 in enumerate(wl.contexts):
                o_ref, lse_ref = oracle_request(wl, 0, r, step, S0 + step)
                check_close(o[r], lse[r], o_ref, lse_ref, f"{wl.name} step{step} r{r} impl{impl} refresh{refresh}")
    snap, ms = kf.route_snapshot(), model.snapshot()
    for key in ("len", "n_ranges", "part", "slot", "free_head", "rr_cursor"):
        assert snap[key] == ms[key], key
    ses.close()
    return outs


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("refresh", [0, 1, 5])
def test_kept_plan_decode_loop_matches_oracle(impl, refresh):
    # contexts chosen so that within 40 steps: tails cross 16-token tile edges many times, request 1 fills its
    # range at step 3 (128 -> new range, forces a rebuild), request 3 starts with a 1-token tail range, request 4
    # sits one token before a tile edge, and the plan ages past `refresh` (0 = default 128: never, 1: every step)
    wl = Workload("kept_plan", 32, 8, 64, 3, [200, 125, 33, 65, 16, 1])
    _decode_loop(wl, impl, steps=40, refresh=refresh)


@pytest.mark.parametrize("impl", IMPLS)
def test_layer_step_one_launch_equals_append_then_attend(impl):
    # kf_layer_step (append + attend + merge in ONE launch: the new K/V row is written to the pool AND patched into the
    # shared-memory copy of the tail tile) must give the bits of kf_kv_append followed by kf_attend, at every step of a
    # loop whose tails cross tile edges, fill ranges and sit in 1-token ranges; and it matches the oracle
    wl = Workload("one_launch", 32, 8, 64, 3, [200, 125, 33, 65, 16, 1])
    a = _decode_loop(wl, impl, steps=40, refresh=0, one_launch=True)
    b = _decode_loop(wl, impl, steps=40, refresh=0, one_launch=False, check_every=40)
    for step, ((oa, la), (ob, lb)) in enumerate(zip(a, b)):
        assert np.array_equal(oa, ob) and np.array_equal(la, lb), step


def test_kept_plan_many_pieces_and_unfused():
    # min_tiles = 1: every tile its own piece, so the stretched level-0 chunk sits among many small pieces
    wl = Workload("kept_plan_pieces", 64, 8, 512, 2, [1500, 700, 511])
    a = _decode_loop(wl, KF_IMPL_TMA, steps=36, refresh=0, fused=True, min_tiles=1, check_every=5)
    b = _decode_loop(wl, KF_IMPL_TMA, steps=36, refresh=0, fused=False, min_tiles=1, check_every=5)
    for (oa, la), (ob, lb) in zip(a, b):     # same plan history => same cuts => bit-identical
        assert np.array_equal(oa, ob) and np.array_equal(la, lb)


def test_attend_after_commit_without_boundary():
    # a commit invalidates the plan on the host side: an attend that follows it without kf_token_boundary rebuilds
    # the plan; if the new position has no route (tail range full) the device reports ESTATE, as before
    wl = Workload("no_boundary", 32, 8, 64, 2, [63, 10])
    ses = Session(wl, steps=4)
    ses.prepare()
    kf = ses.kf
    kf.token_boundary()
    q = ses.q_for(0, 0)
    k_new, v_new = ses.kv_new_for(0, 0)
    ses.layer_step(0, q, k_new, v_new)
    kf.step_commit()                      # len = 63, 10: position 63 still has a route
    q = ses.q_for(0, 1)
    k_new, v_new = ses.kv_new_for(0, 1)
    ses.layer_step(0, q, k_new, v_new)    # no boundary call
    assert kf.status() == KF_OK
    o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
    for r, S0 in enumerate(wl.contexts):
        o_ref, lse_ref = oracle_request(wl, 0, r, 1, S0 + 1)
        check_close(o[r], lse[r], o_ref, lse_ref, f"no_boundary r{r}")
    kf.step_commit()                      # len = 64: request 0 needs a new range, none was opened
    ses.layer_step(0, q, k_new, v_new)
    assert kf.status() == KF_ESTATE
    ses.close()


def test_many_requests_plan_scratch_spills_to_global():
    # 1024 requests x 10 ranges = 10240 (request, range) entries and 4-5 scheduling levels: the plan kernel's
    # per-(level, entry) arrays no longer fit its 192 KB of shared memory and fall back to the global scratch area
    # (kf_state.cu: take()).  Routes against the integer model; sampled requests against the oracle; two steps so
    # that the kept plan is exercised on this path as well.
    import random
    rnd = random.Random(5)
    B, R = 1024, 64
    ctx = [rnd.randrange(560, 640) for _ in range(B)]
    wl = Workload("many_requests", 8, 2, R, 16, ctx)
    ses = Session(wl, steps=2)
    ses.prepare()
    kf = ses.kf
    model = RoutingModel(wl.n_partitions, R, B, kf.Jmax, kf.cfg.slots_per_partition)
    for r, n in enumerate(ses.len0):
        model.open_request(r, n)
    for step in range(2):
        kf.token_boundary()
        model.token_boundary()
        q = ses.q_for(0, step)
        k_new, v_new = ses.kv_new_for(0, step)
        ses.o.fill_(float("nan"))
        ses.lse.fill_(float("nan"))
        ses.layer_step(0, q, k_new, v_new)
        info = kf.plan_info()             # (before the commit: afterwards the plan of the NEXT step would be built)
        assert info["n_entries"] >= 9 * B and info["n_units"] == 2 * info["n_entries"]
        kf.step_commit()
        model.step_commit()
        assert kf.status() == KF_OK
        o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
        assert np.isfinite(o).all() and np.isfinite(lse).all()
        for r in (0, 1, 511, 777, 1023):
            o_ref, lse_ref = oracle_request(wl, 0, r, step, ctx[r] + step)
            check_close(o[r], lse[r], o_ref, lse_ref, f"many_requests step{step} r{r}")
    snap, ms = kf.route_snapshot(), model.snapshot()
    for key in ("len", "n_ranges", "part", "slot", "free_head", "rr_cursor"):
        assert snap[key] == ms[key], key
    ses.close()
