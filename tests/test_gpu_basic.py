"""GPU parity tests (through the C ABI): generator twin, routing / slots / appended bytes bit-exact against
the integer model, attention against the fp64 oracle on small configs (both kernels, fused and unfused)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from conftest import load_golden  # noqa: E402
from kf_inputs import gen, gen_device, workloads  # noqa: E402
from kf_inputs.workloads import Workload  # noqa: E402
from kf_testlib import check_close, host_kv, oracle_request  # noqa: E402
from oracle.routing import RoutingModel  # noqa: E402
from paper_2606_29207_b200 import (KF_ENOSPC, KF_ESTATE, KF_IMPL_SIMPLE, KF_IMPL_TMA, KF_OK, KFlume,  # noqa: E402
                                   make_config)
from paper_2606_29207_b200.workload import Session  # noqa: E402

IMPLS = [KF_IMPL_SIMPLE, KF_IMPL_TMA]


# ------------------------------------------------------------------------------------------------------
def test_generator_device_twin_bit_exact():
    for (stream, layer, req, p0, n, heads) in [(gen.STREAM_K, 0, 0, 0, 300, 8), (gen.STREAM_V, 3, 17, 1000000, 257, 8),
                                               (gen.STREAM_Q, 31, 127, 63, 1, 64)]:
        dev = gen_device.fill(stream, layer, req, p0, n, heads).cpu().numpy()
        host = gen.tensor(stream, layer, req, np.arange(p0, p0 + n), heads)
        assert np.array_equal(dev.view(np.uint16), host.view(np.uint16))
    pos = torch.tensor([5, -1, 70000], dtype=torch.int32, device="cuda")
    rows = gen_device.fill_rows(gen.STREAM_K, 2, pos, 8).cpu().numpy()
    assert np.array_equal(rows[0].view(np.uint16), gen.gen_k(2, 0, [5], 8)[:, 0].view(np.uint16))
    assert np.array_equal(rows[2].view(np.uint16), gen.gen_k(2, 2, [70000], 8)[:, 0].view(np.uint16))
    assert not rows[1].any()


# ------------------------------------------------------------------------------------------------------
def _model_snapshot_equal(kf, model):
    snap = kf.route_snapshot()
    ms = model.snapshot()
    for key in ("len", "n_ranges", "part", "slot", "free_head", "rr_cursor"):
        assert snap[key] == ms[key], key


def _pool_row(kf, part, layer, slot, g, tok, is_v):
    off = kf.pool_offset(layer, slot, g, tok, is_v)
    return kf.pools[part][off:off + 256].cpu().numpy().view(np.uint16)


def test_routing_tiny_scenario_and_appended_bytes():
    g = load_golden("appendix_c_routing.json")["tiny"]
    P, R, lens = g["P"], g["R"], g["load_lens"]
    wl = Workload("tiny", 8, 2, R, P, [n + 1 for n in lens])
    cfg = make_config(8, 2, R, P, 3, 8, 8, n_layers=2)
    kf = KFlume(cfg)
    model = RoutingModel(P, R, 3, 8, 8)
    for r, n in enumerate(lens):
        kf.open_request(r, n)
        model.open_request(r, n)
        for layer in range(2):
            if n:
                k = torch.from_numpy(gen.gen_k(layer, r, np.arange(n), 2)).cuda()
                v = torch.from_numpy(gen.gen_v(layer, r, np.arange(n), 2)).cuda()
                kf.load_context(layer, r, 0, k, v)
    _model_snapshot_equal(kf, model)
    snap = kf.route_snapshot()
    assert [[[p, s] for p, s in zip(snap["part"][r], snap["slot"][r]) if p >= 0] for r in range(3)] == \
        g["after_load"]["routes"]
    for step, st in enumerate(g["steps"]):
        kf.token_boundary()
        ev = model.token_boundary()
        assert [[r, p, s] for (r, _, p, s) in ev] == st["opens"]
        _model_snapshot_equal(kf, model)
        for layer in range(2):
            pos = [model.len[r] for r in range(3)]
            kn = np.stack([gen.gen_k(layer, r, [pos[r]], 2)[:, 0] for r in range(3)])
            vn = np.stack([gen.gen_v(layer, r, [pos[r]], 2)[:, 0] for r in range(3)])
            kf.kv_append(layer, torch.from_numpy(kn).cuda(), torch.from_numpy(vn).cuda())
        for r in range(3):
            p, s, off = model.append_position(r)
            assert [p, s, off] == st["append"][r]
        kf.step_commit()
        model.step_commit()
        assert kf.status() == KF_OK
        _model_snapshot_equal(kf, model)
        assert kf.route_snapshot()["len"] == st["lens_after"]
    # every logical token of every request / layer / head sits, bit-exact, where the model says
    for layer in range(2):
        for r in range(3):
            n = model.len[r]
            K, V = gen.gen_k(layer, r, np.arange(n), 2), gen.gen_v(layer, r, np.arange(n), 2)
            for pos in range(n):
                p, s, off = model.locate(r, pos)
                for hd in range(2):
                    assert np.array_equal(_pool_row(kf, p, layer, s, hd, off, False), K[hd, pos].view(np.uint16))
                    assert np.array_equal(_pool_row(kf, p, layer, s, hd, off, True), V[hd, pos].view(np.uint16))
    kf.close()


def test_close_reuse_and_errors():
    cfg = make_config(8, 2, 4, 2, 3, 4, 4)
    kf = KFlume(cfg)
    m = RoutingModel(2, 4, 3, 4, 4)
    for (r, n) in [(0, 8), (1, 4)]:
        kf.open_request(r, n)
        m.open_request(r, n)
    kf.close_request(0)
    m.close_request(0)
    kf.open_request(2, 8)
    m.open_request(2, 8)
    _model_snapshot_equal(kf, m)
    assert kf.status() == KF_OK
    kf.open_request(1, 4)                      # already open
    assert kf.status() == KF_ESTATE
    assert kf.status() == KF_OK                # cleared
    kf.close_request(0)                        # not open
    assert kf.status() == KF_ESTATE
    kf.close()
    # ENOSPC: partition full
    kf = KFlume(make_config(8, 2, 4, 1, 1, 8, 2))
    kf.open_request(0, 8)
    assert kf.status() == KF_OK
    kf.token_boundary()
    assert kf.status() == KF_ENOSPC
    kf.close()
    # ESTATE: append / attend without a route for the tail position
    kf = KFlume(make_config(8, 2, 4, 2, 1, 8, 4))
    kf.open_request(0, 4)
    z = torch.zeros((1, 2, 128), dtype=torch.float16, device="cuda")
    kf.kv_append(0, z, z)
    assert kf.status() == KF_ESTATE
    kf.close()


# ------------------------------------------------------------------------------------------------------
def _run_and_check(wl, impl, fused, check_partials=True, heads=None, reqs=None, min_tiles=0, scale=0.0, mutate=None):
    ses = Session(wl, impl=impl, min_tiles=min_tiles, softmax_scale=scale)
    ses.prepare()
    kf = ses.kf
    kf.token_boundary()
    q = ses.q_for(0, 0)
    k_new, v_new = ses.kv_new_for(0, 0)
    if mutate is not None:
        mutate(ses, q, k_new, v_new)
    ses.o.fill_(float("nan"))
    ses.lse.fill_(float("nan"))
    ses.o_part.fill_(float("nan"))
    ses.lse_part.fill_(float("nan"))
    ses.layer_step(0, q, k_new, v_new, fused=fused, want_partials=True)
    assert kf.status() == KF_OK
    o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
    op, lp = ses.o_part.cpu().numpy(), ses.lse_part.cpu().numpy()
    out = {"o": o, "lse": lse, "o_part": op, "lse_part": lp, "ses": ses}
    if mutate is None:
        for r in (range(wl.batch) if reqs is None else reqs):
            S = wl.contexts[r]
            hs = list(range(wl.n_q_heads)) if heads is None else heads
            o_ref, lse_ref, op_ref, lp_ref = oracle_request(wl, 0, r, 0, S, hs, scale or None, ranges=True)
            check_close(o[r][hs], lse[r][hs], o_ref, lse_ref, f"{wl.name} r{r} impl{impl} fused{fused}")
            if check_partials:
                J = op_ref.shape[0]
                for j in range(J):
                    check_close(op[r, j][hs], lp[r, j][hs], op_ref[j], lp_ref[j], f"{wl.name} r{r} range{j}")
                assert np.isnan(lp[r, J:]).all()          # rows of non-existent ranges untouched
    return out


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("fused", [True, False])
def test_t0_tiny_golden(impl, fused):
    wl = workloads.tiny_t0()
    out = _run_and_check(wl, impl, fused)
    g = load_golden("appendix_b_t0.json")
    assert np.abs(out["lse"][0] - np.array(g["lse"])).max() < 1e-4
    assert np.abs(out["o"][0][:, 0] - np.array(g["o_col0"])).max() < 2e-3
    assert np.abs(out["lse_part"][0, 1] - np.array(g["lse_range1"])).max() < 1e-4
    # 1-token range: o = V exactly
    V = gen.gen_v(0, 0, [4], 2)
    for h in range(8):
        assert np.array_equal(out["o_part"][0, 1, h], V[h // 4, 0].astype(np.float32))
    out["ses"].close()


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("fused", [True, False])
def test_cfg1(impl, fused):
    wl = workloads.cfg1()
    out = _run_and_check(wl, impl, fused)
    g = load_golden("appendix_b_cfg1.json")
    for hs, e in g["heads"].items():
        h = int(hs)
        assert abs(out["lse"][0, h] - e["lse"]) < 1e-4 * e["lse"]
        assert abs(out["lse_part"][0, 0, h] - e["lse_r0"]) < 1e-4 * e["lse_r0"]
        assert abs(out["o"][0, h, 64] - e["o64"]) < 2e-3
    out["ses"].close()


RAGGED = [
    # name, Hq, Hkv, R, P, contexts
    ("one_token", 8, 2, 16, 2, [1]),
    ("ragged_small", 32, 8, 64, 3, [1, 2, 15, 16, 17, 63, 64, 65, 100, 129]),
    ("ragged_mid", 32, 8, 256, 4, [1000, 257, 256, 255, 513, 31, 2049]),
    ("g8", 64, 8, 128, 2, [300, 129, 77]),
    ("g1_mha", 8, 8, 128, 2, [200, 31]),
    ("g2", 16, 8, 32, 2, [97]),
    ("g6", 48, 8, 128, 3, [150, 400]),
    ("small_R", 8, 2, 4, 2, [23, 9, 4, 5]),
    ("R1", 8, 2, 1, 3, [7]),
]


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("case", RAGGED, ids=[c[0] for c in RAGGED])
def test_ragged_shapes_fused_and_unfused(impl, case):
    name, Hq, Hkv, R, P, ctx = case
    wl = Workload(name, Hq, Hkv, R, P, ctx)
    a = _run_and_check(wl, impl, True)
    b = _run_and_check(wl, impl, False)
    # fused and unfused paths reduce in the same order: bit-identical
    assert np.array_equal(a["o"], b["o"]) and np.array_equal(a["lse"], b["lse"])
    for r, S in enumerate(ctx):
        J = -(-S // R)
        assert np.array_equal(a["o_part"][r, :J], b["o_part"][r, :J])
    a["ses"].close()
    b["ses"].close()


@pytest.mark.parametrize("impl", IMPLS)
def test_many_workers_per_unit(impl):
    # min_tiles=1 -> every 16-token tile its own piece: stresses piece buffers and the 2-level fused merge
    wl = Workload("split_hard", 32, 8, 512, 2, [1500, 700])
    a = _run_and_check(wl, impl, True, min_tiles=1)
    info = a["ses"].kf.plan_info()
    assert info["n_pieces"] > info["n_units"]
    b = _run_and_check(wl, impl, False, min_tiles=1)
    assert np.array_equal(a["o"], b["o"]) and np.array_equal(a["lse"], b["lse"])
    a["ses"].close()
    b["ses"].close()


def test_kernels_agree():
    wl = Workload("agree", 32, 8, 256, 4, [1000, 257, 31])
    a = _run_and_check(wl, KF_IMPL_SIMPLE, True)
    b = _run_and_check(wl, KF_IMPL_TMA, True)
    assert np.abs(a["o"] - b["o"]).max() < 6e-4 and np.abs(a["lse"] - b["lse"]).max() < 1e-4  # P is fp16 in the TMA kernel
    a["ses"].close()
    b["ses"].close()


@pytest.mark.parametrize("impl", IMPLS)
def test_partition_mask_subsets(impl):
    wl = Workload("mask", 32, 8, 128, 4, [700, 130, 300])
    ses = Session(wl, impl=impl)
    ses.prepare()
    kf = ses.kf
    kf.token_boundary()
    q = ses.q_for(0, 0)
    k_new, v_new = ses.kv_new_for(0, 0)
    kf.kv_append(0, k_new, v_new)
    full_o, full_l = torch.zeros_like(ses.o_part), torch.zeros_like(ses.lse_part)
    kf.partial_attend(0, q, full_o, full_l)
    acc_o = torch.full_like(full_o, float("nan"))
    acc_l = torch.full_like(full_l, float("nan"))
    snap = kf.route_snapshot()
    for p in range(4):
        mask = [1 if i == p else 0 for i in range(4)]
        kf.partial_attend(0, q, acc_o, acc_l, partition_mask=mask)
        # rows of other partitions untouched so far
        for r in range(3):
            for j in range(snap["n_ranges"][r]):
                done = snap["part"][r][j] <= p
                assert bool(torch.isnan(acc_l[r, j]).any().item()) == (not done)
    for r in range(3):
        J = snap["n_ranges"][r]
        assert torch.equal(acc_o[r, :J], full_o[r, :J]) and torch.equal(acc_l[r, :J], full_l[r, :J])
    # merge of the accumulated partials == fused result
    kf.merge_partials(acc_o, acc_l, ses.o, ses.lse)
    o1, l1 = ses.o.clone(), ses.lse.clone()
    kf.attend(0, q, ses.o, ses.lse)
    assert torch.equal(o1, ses.o) and torch.equal(l1, ses.lse)
    assert kf.status() == KF_OK
    ses.close()


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("where", ["first", "tile_edge", "range_last", "tail"])
def test_peaked_softmax(impl, where):
    """One key = 4*q_h: weight ~ 1 on one token, |o| ~ 1 -> the absolute tolerance is meaningful."""
    R, S = 64, 200
    wl = Workload("peaked", 8, 2, R, 2, [S])
    tstar = {"first": 0, "tile_edge": 16, "range_last": R - 1, "tail": S - 1}[where]
    h = 5
    q_np = gen.gen_q(0, 0, 0, 8)
    K, V = host_kv(wl, 0, 0, S)
    K = K.copy()
    K[h // 4, tstar] = (q_np[h].astype(np.float32) * 4).astype(np.float16)

    ses = Session(wl, impl=impl)
    ses.open_all()
    kf = ses.kf
    kt, vt = torch.from_numpy(K).cuda(), torch.from_numpy(V).cuda()
    kf.load_context(0, 0, 0, kt[:, :S - 1].contiguous(), vt[:, :S - 1].contiguous())
    kf.token_boundary()
    q = ses.q_for(0, 0)
    kf.kv_append(0, kt[:, S - 1].contiguous().view(1, 2, 128), vt[:, S - 1].contiguous().view(1, 2, 128))
    kf.attend(0, q, ses.o, ses.lse)
    assert kf.status() == KF_OK
    o_ref, lse_ref = oracle.attend(q_np, K, V)
    assert np.abs(o_ref[h] - V[h // 4, tstar].astype(np.float64)).max() < 1e-6   # the oracle itself is peaked
    check_close(ses.o[0].cpu().numpy(), ses.lse[0].cpu().numpy(), o_ref, lse_ref, f"peaked {where}")
    ses.close()


@pytest.mark.parametrize("impl", IMPLS)
def test_gqa_mapping_on_device(impl):
    wl = Workload("gqa", 8, 2, 64, 2, [150])
    base = _run_and_check(wl, impl, True)

    def same_q(ses, q, k_new, v_new):
        q[0, :] = q[0, 0]
    a = _run_and_check(wl, impl, True, mutate=same_q)
    o = a["o"][0]
    assert np.array_equal(o[1], o[0]) and np.array_equal(o[3], o[0]) and np.array_equal(o[5], o[4])
    assert not np.array_equal(o[0], o[4])

    def poison_kv1(ses, q, k_new, v_new):
        # overwrite kv head 1 of the whole context: heads 0..3 must stay bit-identical
        n = ses.len0[0]
        kf = ses.kf
        K = gen_device.fill(gen.STREAM_K, 9, 0, 0, n, 2)
        V = gen_device.fill(gen.STREAM_V, 9, 0, 0, n, 2)
        K0 = gen_device.fill(gen.STREAM_K, 0, 0, 0, n, 2)
        V0 = gen_device.fill(gen.STREAM_V, 0, 0, 0, n, 2)
        K[0], V[0] = K0[0], V0[0]
        kf.load_context(0, 0, 0, K, V)
    b = _run_and_check(wl, impl, True, mutate=poison_kv1)
    assert np.array_equal(b["o"][0][:4], base["o"][0][:4]) and np.array_equal(b["lse"][0][:4], base["lse"][0][:4])
    assert not np.array_equal(b["o"][0][4:], base["o"][0][4:])
    for x in (base, a, b):
        x["ses"].close()


def test_custom_scale_and_run_to_run_determinism():
    wl = Workload("scale", 32, 8, 128, 2, [333, 90])
    a = _run_and_check(wl, KF_IMPL_TMA, True, scale=0.05)
    b = _run_and_check(wl, KF_IMPL_TMA, True, scale=0.05, min_tiles=0)
    assert np.array_equal(a["o"], b["o"]) and np.array_equal(a["lse"], b["lse"])
    ses = a["ses"]
    q = ses.q_for(0, 0)
    for _ in range(5):
        o2, l2 = torch.zeros_like(ses.o), torch.zeros_like(ses.lse)
        ses.kf.attend(0, q, o2, l2)
        assert torch.equal(o2, ses.o) and torch.equal(l2, ses.lse)
    a["ses"].close()
    b["ses"].close()


def test_layer_step_host_matches_device_path():
    wl = Workload("host", 32, 8, 128, 2, [300, 45, 129])
    ses = Session(wl)
    ses.prepare()
    kf = ses.kf
    kf.token_boundary()
    q = ses.q_for(0, 0)
    k_new, v_new = ses.kv_new_for(0, 0)
    ses.layer_step(0, q, k_new, v_new)
    o_dev, l_dev = ses.o.cpu(), ses.lse.cpu()
    qh, kh, vh = q.cpu().pin_memory(), k_new.cpu().pin_memory(), v_new.cpu().pin_memory()
    oh = torch.zeros((3, 32, 128), dtype=torch.float32).pin_memory()
    lh = torch.zeros((3, 32), dtype=torch.float32).pin_memory()
    kf.layer_step_host(0, qh, kh, vh, oh, lh)
    torch.cuda.synchronize()
    assert torch.equal(oh, o_dev) and torch.equal(lh, l_dev)
    assert kf.status() == KF_OK
    ses.close()


@pytest.mark.parametrize("impl", IMPLS)
def test_closed_request_rows_untouched_and_64_partitions(impl):
    # P = 64 (the maximum), 5 requests of which #1 and #3 are closed before the step: their output rows must stay
    # untouched, the others must match the oracle; the freed slots are reused by a request opened afterwards
    wl = Workload("holes", 32, 8, 32, 64, [100, 70, 33, 64, 129])
    ses = Session(wl, impl=impl, slack_slots=2)
    ses.prepare()
    kf = ses.kf
    kf.close_request(1)
    kf.close_request(3)
    kf.token_boundary()
    q = ses.q_for(0, 0)
    k_new, v_new = ses.kv_new_for(0, 0)
    ses.o.fill_(float("nan"))
    ses.lse.fill_(float("nan"))
    ses.layer_step(0, q, k_new, v_new)
    assert kf.status() == KF_OK
    o, lse = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
    for r in (0, 2, 4):
        o_ref, lse_ref = oracle_request(wl, 0, r, 0, wl.contexts[r])
        check_close(o[r], lse[r], o_ref, lse_ref, f"holes r{r}")
    for r in (1, 3):
        assert np.isnan(o[r]).all() and np.isnan(lse[r]).all()
    snap = kf.route_snapshot()
    assert snap["len"][1] == -1 and snap["n_ranges"][3] == 0
    ses.close()
