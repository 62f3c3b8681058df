"""GPU tests of slot exhaustion (readings 10 and 24): a full partition is passed over by the round-robin,
a request whose token boundary finds no slot waits -- no append, no commit -- and resumes, bit-exact against the
integer model, as soon as a slot is freed or a node is activated; attention after the resume matches the fp64 oracle."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from kf_inputs import gen  # noqa: E402
from kf_testlib import check_close  # noqa: E402
from oracle.routing import RoutingError, RoutingModel  # noqa: E402
from paper_2606_29207_b200 import KF_ENOSPC, KF_IMPL_SIMPLE, KF_IMPL_TMA, KF_OK, KFlume, make_config  # noqa: E402

HQ, HKV = 8, 2


def _same(kf, model):
    snap, ms = kf.route_snapshot(), model.snapshot()
    for key in ("len", "n_ranges", "part", "slot", "free_head", "rr_cursor"):
        assert snap[key] == ms[key], key


def _open(kf, model, r, n):
    kf.open_request(r, n)
    model.open_request(r, n)
    if n:
        pos = np.arange(n)
        kf.load_context(0, r, 0, torch.from_numpy(gen.gen_k(0, r, pos, HKV)).cuda(),
                        torch.from_numpy(gen.gen_v(0, r, pos, HKV)).cuda())


def _step(kf, model, step, o, lse, expect_enospc):
    """One decode step on device and model; rows of k_new / v_new are the generator's values at each request's
    CURRENT position (a waiting request presents the same token again).  Returns the requests that attended the
    whole context (those with a route for their tail position)."""
    B = model.B
    kf.token_boundary()
    try:
        model.token_boundary()
        failed = False
    except RoutingError:
        failed = True
    assert failed == expect_enospc
    _same(kf, model)
    kn = np.zeros((B, HKV, 128), np.float16)
    vn = np.zeros((B, HKV, 128), np.float16)
    q = np.zeros((B, HQ, 128), np.float16)
    served = []
    for r in range(B):
        if model.len[r] < 0:
            continue
        kn[r] = gen.gen_k(0, r, [model.len[r]], HKV)[:, 0]
        vn[r] = gen.gen_v(0, r, [model.len[r]], HKV)[:, 0]
        q[r] = gen.gen_q(0, r, step, HQ)
        if len(model.route[r]) * model.R > model.len[r]:
            served.append(r)
    kf.kv_append(0, torch.from_numpy(kn).cuda(), torch.from_numpy(vn).cuda())
    kf.attend(0, torch.from_numpy(q).cuda(), o, lse)
    kf.step_commit()
    # ENOSPC from the boundary is latched first; the append / plan of a waiting request add ESTATE behind it
    assert kf.status() == (KF_ENOSPC if expect_enospc else KF_OK)
    oh, lh = o.cpu().numpy(), lse.cpu().numpy()
    for r in served:
        n = model.len[r] + 1
        pos = np.arange(n)
        o_ref, lse_ref = oracle.attend(q[r], gen.gen_k(0, r, pos, HKV), gen.gen_v(0, r, pos, HKV))
        check_close(oh[r], lh[r], o_ref, lse_ref, f"step{step} r{r}")
    # a waiting request is still answered, over the tokens it has committed (kflume.h, kf_token_boundary) -- step after
    # step, whether the work plan was rebuilt at this boundary or kept (a failed allocation changes no route)
    for r in range(B):
        if model.len[r] > 0 and r not in served:
            pos = np.arange(model.len[r])
            o_ref, lse_ref = oracle.attend(q[r], gen.gen_k(0, r, pos, HKV), gen.gen_v(0, r, pos, HKV))
            check_close(oh[r], lh[r], o_ref, lse_ref, f"step{step} waiting r{r}")
    model.step_commit()
    _same(kf, model)
    return served


@pytest.mark.parametrize("refresh", [0, 1])     # 0: the plan is kept while nothing changes; 1: rebuilt at every boundary
@pytest.mark.parametrize("impl", [KF_IMPL_SIMPLE, KF_IMPL_TMA])
def test_request_waits_for_a_slot_and_resumes(impl, refresh):
    # one node, 3 slots, R = 4: r0 (4 tokens) and r1 (8 tokens) fill it; both tail ranges are full
    cfg = make_config(HQ, HKV, 4, 1, 3, 4, 3, attend_impl=impl, plan_refresh_steps=refresh)
    kf = KFlume(cfg)
    model = RoutingModel(1, 4, 3, 4, 3)
    _open(kf, model, 0, 4)
    _open(kf, model, 1, 8)
    o = torch.zeros((3, HQ, 128), dtype=torch.float32, device="cuda")
    lse = torch.zeros((3, HQ), dtype=torch.float32, device="cuda")
    for step in range(3):                                  # nobody can move: lengths stay, nothing is appended
        assert _step(kf, model, step, o, lse, expect_enospc=True) == []
        assert model.len == [4, 8, -1]
    kf.close_request(1)
    model.close_request(1)
    for step in range(3, 9):                # r0 takes the slot freed last (LIFO), fills it at 8, takes the other one
        assert _step(kf, model, step, o, lse, expect_enospc=False) == [0]
    assert model.len[0] == 10 and model.route[0] == [(0, 0), (0, 2), (0, 1)]
    kf.close()


def test_full_partition_is_passed_over_after_scale_down():
    # 2 nodes x 2 slots, R = 4.  With only node 0 active two requests fill it; node 1 joins; the round-robin now
    # passes over the full node 0 for every new range until node 1 is full too (ENOSPC), and a waiting request
    # resumes when a request on node 0 leaves.
    cfg = make_config(HQ, HKV, 4, 2, 4, 4, 2)
    kf = KFlume(cfg)
    model = RoutingModel(2, 4, 4, 4, 2)
    kf.set_active_partitions([1, 0])
    model.set_active([1, 0])
    _open(kf, model, 0, 3)
    _open(kf, model, 1, 2)
    kf.set_active_partitions([1, 1])
    model.set_active([1, 1])
    _same(kf, model)
    o = torch.zeros((4, HQ, 128), dtype=torch.float32, device="cuda")
    lse = torch.zeros((4, HQ), dtype=torch.float32, device="cuda")
    step = 0
    _step(kf, model, step, o, lse, False)                  # r0 -> 4
    step += 1
    assert _step(kf, model, step, o, lse, False) == [0, 1]  # r0 opens its 2nd range on node 1: (1,0)
    assert model.route[0] == [(0, 0), (1, 0)]
    step += 1
    assert _step(kf, model, step, o, lse, False) == [0, 1]  # r1 at 4: node 0 is full -> passed over -> (1,1)
    assert model.route[1] == [(0, 1), (1, 1)]
    for _ in range(2):
        step += 1
        _step(kf, model, step, o, lse, False)
    # r0 at 8: needs a third range, everything is full -> waits; r1 (at 7) still moves
    step += 1
    assert _step(kf, model, step, o, lse, True) == [1]
    assert model.len[:2] == [8, 8]
    step += 1
    assert _step(kf, model, step, o, lse, True) == []      # now both wait
    kf.close_request(1)
    model.close_request(1)
    step += 1
    assert _step(kf, model, step, o, lse, False) == [0]    # r0 resumes on the slot r1 left behind on node 0
    assert model.len[0] == 9 and model.route[0] == [(0, 0), (1, 0), (0, 1)]
    kf.close()
