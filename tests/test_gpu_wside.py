"""GPU parity of the W-node stages (kf_w_project_q / _kv, kf_w_post_attention: the tcgen05 GEMMs of kf_wgemm.cu) and of
the M = 2 inter-layer pipeline (kf_pipeline_step) against the fp64 oracle (oracle/wside.py + oracle.attend), on seeded
synthetic weights and hidden states.  Tolerances: a stored fp16 value may differ from the fp64
value by half an ulp (2^-11 relative) plus what one-ulp differences in the fp16 operands of the previous stage add."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from kf_inputs import gen, gen_device  # noqa: E402
from kf_inputs.workloads import Workload  # noqa: E402
from oracle import wside as ow  # noqa: E402
from paper_2606_29207_b200 import KF_OK, KF_W_DOWN, KF_W_GATE, KF_W_KV, KF_W_O, KF_W_Q, KF_W_UP  # noqa: E402
from paper_2606_29207_b200.workload import W_STREAMS, Session, make_wside  # noqa: E402


def _close(got, ref, what, rel=1.5e-3, rms_frac=1.5e-3):
    got, ref = np.asarray(got, np.float64), np.asarray(ref, np.float64)
    assert got.shape == ref.shape, (what, got.shape, ref.shape)
    assert np.isfinite(got).all(), f"{what}: non-finite"
    tol = rel * np.abs(ref) + rms_frac * np.sqrt(np.mean(ref * ref)) + 1e-6
    bad = np.abs(got - ref) > tol
    assert not bad.any(), f"{what}: {bad.sum()} of {bad.size} outside tolerance, max err {np.abs(got - ref).max():.3e}"
    return float(np.abs(got - ref).max())


def _host_weights(w, layer, rows=None):
    return {which: gen.gen_weight(stream, layer, *w.shape(which)) for which, stream in W_STREAMS.items()}


@pytest.mark.parametrize("batch", [1, 7, 16, 33, 64, 100, 128])
def test_every_contraction_vs_oracle(batch):
    # hidden 512, 4 query / 2 KV heads, ffn 1024, two layers: every tile count, split-K choice and batch padding of the
    # kernel (NB = 16, 32, 64, 128; rows >= batch are zero-filled by TMA and never stored)
    hidden, Hq, Hkv, ffn = 512, 4, 2, 1024
    w = make_wside(hidden, Hq, Hkv, ffn, n_layers=2, max_batch=128)
    for layer in (0, 1):
        W = _host_weights(w, layer)
        for which in W:                                   # the device twin filled exactly these bits
            assert np.array_equal(w.weight(layer, which).cpu().numpy().view(np.uint16), W[which].view(np.uint16))
        x = gen_device.fill_x(layer, batch, 3, hidden)
        xh = gen.gen_x(layer, batch, 3, hidden)
        assert np.array_equal(x.cpu().numpy().view(np.uint16), xh.view(np.uint16))
        q = torch.full((batch, Hq, 128), float("nan"), dtype=torch.float16, device="cuda")
        k = torch.full((batch, Hkv, 128), float("nan"), dtype=torch.float16, device="cuda")
        v = torch.full_like(k, float("nan"))
        w.project_q(layer, x, q)
        w.project_kv(layer, x, k, v)
        ref = ow.project(xh, W[KF_W_Q], W[KF_W_KV])
        _close(q.cpu().numpy().reshape(batch, -1), ref["q"], f"q layer{layer} B{batch}")
        _close(k.cpu().numpy().reshape(batch, -1), ref["k"], f"k layer{layer} B{batch}")
        _close(v.cpu().numpy().reshape(batch, -1), ref["v"], f"v layer{layer} B{batch}")
        # post-attention on a seeded "attention output" (unit-variance values of the q stream, as fp32)
        o_h = gen.tensor(gen.STREAM_Q, layer + 7, 0, np.arange(batch), Hq).transpose(1, 0, 2).astype(np.float32)
        o = torch.from_numpy(np.ascontiguousarray(o_h)).cuda()
        xn = torch.full((batch, hidden), float("nan"), dtype=torch.float16, device="cuda")
        w.post_attention(layer, o, xn)
        refp = ow.post_attention(o_h.reshape(batch, -1), W[KF_W_O], W[KF_W_GATE], W[KF_W_UP], W[KF_W_DOWN])
        _close(xn.cpu().numpy(), refp["x"], f"x' layer{layer} B{batch}", rel=4e-3, rms_frac=4e-3)
    # run to run: bit-identical (split-K partial sums are added in split order)
    xn2 = torch.empty_like(xn)
    w.post_attention(1, o, xn2)
    assert torch.equal(xn, xn2)
    w.close()


def test_llama_8b_layer_shape_sampled_rows():
    # the shape the paper serves (Llama-3.1-8B: hidden 4096, 32/8 heads, ffn 14336), one layer, batch 64; the oracle
    # evaluates 3 batch rows (rows are independent in every stage)
    hidden, Hq, Hkv, ffn, batch = 4096, 32, 8, 14336, 64
    w = make_wside(hidden, Hq, Hkv, ffn, n_layers=1, max_batch=batch)
    rows = [0, 31, 63]
    W = {which: w.weight(0, which).cpu().numpy() for which in W_STREAMS}       # device twin == gen.py: tested above
    spot = gen.gen_weight(gen.STREAM_WDOWN, 0, 2, ffn)
    assert np.array_equal(W[KF_W_DOWN][:2].view(np.uint16), spot.view(np.uint16))
    x = gen_device.fill_x(0, batch, 0, hidden)
    xh = x.cpu().numpy()
    q = torch.empty((batch, Hq, 128), dtype=torch.float16, device="cuda")
    k = torch.empty((batch, Hkv, 128), dtype=torch.float16, device="cuda")
    v = torch.empty_like(k)
    w.project_q(0, x, q)
    w.project_kv(0, x, k, v)
    ref = ow.project(xh[rows], W[KF_W_Q], W[KF_W_KV])
    _close(q.cpu().numpy().reshape(batch, -1)[rows], ref["q"], "8B q")
    _close(k.cpu().numpy().reshape(batch, -1)[rows], ref["k"], "8B k")
    _close(v.cpu().numpy().reshape(batch, -1)[rows], ref["v"], "8B v")
    o_h = gen.tensor(gen.STREAM_Q, 9, 0, np.arange(batch), Hq).transpose(1, 0, 2).astype(np.float32)
    o = torch.from_numpy(np.ascontiguousarray(o_h)).cuda()
    xn = torch.empty((batch, hidden), dtype=torch.float16, device="cuda")
    w.post_attention(0, o, xn)
    refp = ow.post_attention(o_h.reshape(batch, -1)[rows], W[KF_W_O], W[KF_W_GATE], W[KF_W_UP], W[KF_W_DOWN])
    _close(xn.cpu().numpy()[rows], refp["x"], "8B x'", rel=4e-3, rms_frac=4e-3)
    w.close()


def _oracle_layer(wl, W, layer, x16, step, lens):
    """One decode layer of the oracle: project, append to the generator's context, attend, post.  Returns x' (fp16)."""
    B = x16.shape[0]
    p = ow.project(x16, W[KF_W_Q], W[KF_W_KV])
    o = np.zeros((B, wl.n_q_heads * 128))
    for r in range(B):
        n = lens[r]
        pos = np.arange(n)
        K = np.concatenate([gen.gen_k(layer, r, pos, wl.n_kv_heads, wl.seed), p["k16"][r].reshape(wl.n_kv_heads, 1, 128)], 1)
        V = np.concatenate([gen.gen_v(layer, r, pos, wl.n_kv_heads, wl.seed), p["v16"][r].reshape(wl.n_kv_heads, 1, 128)], 1)
        o_r, _ = oracle.attend(p["q16"][r].reshape(wl.n_q_heads, 128), np.ascontiguousarray(K), np.ascontiguousarray(V))
        o[r] = o_r.reshape(-1)
    return ow.post_attention(o, W[KF_W_O], W[KF_W_GATE], W[KF_W_UP], W[KF_W_DOWN])["x16"]


def test_pipeline_step_serial_equals_pipelined_and_matches_oracle_chain():
    # two microbatches (different requests, own routing tables and pools), two layers, two decode steps.  The hidden
    # state of layer l+1 is the x' of layer l, the appended K/V rows are the projected ones: the whole decode layer
    # chain proj -> append -> attend -> merge -> W_O -> FFN, against the oracle chain on the same seeded inputs.
    hidden, Hq, Hkv, ffn, L = 512, 8, 2, 1024, 2
    w = make_wside(hidden, Hq, Hkv, ffn, n_layers=L, max_batch=16)
    Wh = [_host_weights(w, l) for l in range(L)]
    wls = [Workload("mb0", Hq, Hkv, 64, 2, [200, 64, 33, 1], n_layers=L),
           Workload("mb1", Hq, Hkv, 64, 2, [129, 17, 300], n_layers=L, seed=gen.SEED + 1)]
    steps = 2
    outs = {}
    for mode in (0, 1):
        sess = [Session(wl, steps=steps, n_layers_phys=L, attend_sms=64 if mode else 0) for wl in wls]
        for s in sess:
            s.prepare()
        ws, as_ = torch.cuda.Stream(), torch.cuda.Stream()
        res = []
        with torch.cuda.stream(ws):
            bufs = []
            for wl in wls:
                B = wl.batch
                bufs.append({"q": torch.zeros((B, Hq, 128), dtype=torch.float16, device="cuda"),
                             "k": torch.zeros((B, Hkv, 128), dtype=torch.float16, device="cuda"),
                             "v": torch.zeros((B, Hkv, 128), dtype=torch.float16, device="cuda"),
                             "o": torch.zeros((B, Hq, 128), dtype=torch.float32, device="cuda"),
                             "lse": torch.zeros((B, Hq), dtype=torch.float32, device="cuda")})
            for t in range(steps):
                xs = [gen_device.fill_x(0, wl.batch, t, hidden, seed=wl.seed) for wl in wls]
                ws.synchronize()
                w.pipeline_step([s.kf for s in sess], list(range(L)), xs, [b["q"] for b in bufs], [b["k"] for b in bufs],
                                [b["v"] for b in bufs], [b["o"] for b in bufs], [b["lse"] for b in bufs], mode, ws, as_)
                ws.synchronize()
                as_.synchronize()
                res.append([x.cpu().numpy().copy() for x in xs])
            for s in sess:
                assert s.kf.status() == KF_OK
                assert s.kf.route_snapshot()["len"] == [n + steps for n in s.len0]
        outs[mode] = res
        for s in sess:
            s.close()
    for t in range(steps):
        for m in range(2):
            assert np.array_equal(outs[0][t][m].view(np.uint16), outs[1][t][m].view(np.uint16)), (t, m)
    # oracle chain, step 0 (the context of step 1 would contain the projected rows of step 0 as well)
    for m, wl in enumerate(wls):
        x = gen.gen_x(0, wl.batch, 0, hidden, wl.seed)
        lens = [s - 1 for s in wl.contexts]
        for layer in range(L):
            x = _oracle_layer(wl, Wh[layer], layer, x, 0, lens)
        _close(outs[0][0][m], x.astype(np.float64), f"pipeline chain microbatch {m}", rel=1e-2, rms_frac=1e-2)
    w.close()
