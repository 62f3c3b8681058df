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


# Gates, derived in DESIGN.md section 6 ("Tolerances of the W-side parity tests") from the 2^-11 storage model:
#   one stage (q, k, v):                     1.5e-3 (|ref| + rms)   = 3 u        with u = 2^-11 = 4.9e-4   (seen: 0.73 u)
#   x' behind three stored tensors (o16, y, h) + its own rounding:  2.5e-3 = 5 u                           (seen: 1.5 u)
#   two chained layers incl. attention on projected q / k / v:      1e-2 ~ 20 u                            (seen: 5.4 u)
STAGE_REL, X_REL, CHAIN_REL = 1.5e-3, 2.5e-3, 1e-2


def _close(got, ref, what, rel=STAGE_REL, rms_frac=STAGE_REL):
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
        _close(xn.cpu().numpy(), refp["x"], f"x' layer{layer} B{batch}", rel=X_REL, rms_frac=X_REL)
    # run to run: bit-identical (split-K partial sums are added in split order)
    xn2 = torch.empty_like(xn)
    w.post_attention(1, o, xn2)
    assert torch.equal(xn, xn2)
    w.close()


@pytest.mark.parametrize("sms", [1, 3, 4, 5, 7, 8, 13])
@pytest.mark.parametrize("batch", [16, 128])
def test_span_decompositions_of_the_stream_k_grid(batch, sms):
    # The GEMM cuts the (tile, k-block) sequence into one span per CTA (kf_wgemm.cu), so WHICH tiles are shared between
    # CTAs, which slot a piece lands in and what the fix-up kernel adds all depend on the CTA count.  hidden 512 = 8
    # k-blocks per tile; Wq has 4 tiles, Wkv 4, Wo 4, gate/up 8, down 4 (16 k-blocks).  With 4 or 8 CTAs every span
    # boundary of the 4-tile GEMMs is a tile boundary (no fix-up launch: checked through the launch counter); with 3, 5,
    # 7 and 13 CTAs spans start and end inside tiles (3 CTAs on gate/up: 22 k-blocks per span = the tail of one tile, two
    # whole tiles and the head of a fourth); 1 CTA walks every tile alone.  Everything against the fp64 oracle.
    hidden, Hq, Hkv, ffn = 512, 4, 2, 1024
    w = make_wside(hidden, Hq, Hkv, ffn, n_layers=1, max_batch=128)
    W = _host_weights(w, 0)
    w.set_sms(sms)
    x = gen_device.fill_x(0, batch, 5, hidden)
    xh = gen.gen_x(0, batch, 5, hidden)
    q = torch.full((batch, Hq, 128), float("nan"), dtype=torch.float16, device="cuda")
    k = torch.full((batch, Hkv, 128), float("nan"), dtype=torch.float16, device="cuda")
    v = torch.full_like(k, float("nan"))
    n0 = w.launch_count()
    w.project_q(0, x, q)
    n1 = w.launch_count()
    w.project_kv(0, x, k, v)
    # 4 tiles x 8 k-blocks = 32 pairs: ceil(32 / sms) is a multiple of 8 exactly for sms in {1, 2, 4}; 8 CTAs get 4 each
    assert n1 - n0 == (1 if sms in (1, 4) else 2), (sms, n1 - n0)
    ref = ow.project(xh, W[KF_W_Q], W[KF_W_KV])
    _close(q.cpu().numpy().reshape(batch, -1), ref["q"], f"q sms{sms} B{batch}")
    _close(k.cpu().numpy().reshape(batch, -1), ref["k"], f"k sms{sms} B{batch}")
    _close(v.cpu().numpy().reshape(batch, -1), ref["v"], f"v sms{sms} B{batch}")
    o_h = gen.tensor(gen.STREAM_Q, 11, 0, np.arange(batch), Hq).transpose(1, 0, 2).astype(np.float32)
    o = torch.from_numpy(np.ascontiguousarray(o_h)).cuda()
    xn = torch.full((batch, hidden), float("nan"), dtype=torch.float16, device="cuda")
    w.post_attention(0, o, xn)
    refp = ow.post_attention(o_h.reshape(batch, -1), W[KF_W_O], W[KF_W_GATE], W[KF_W_UP], W[KF_W_DOWN])
    _close(xn.cpu().numpy(), refp["x"], f"x' sms{sms} B{batch}", rel=X_REL, rms_frac=X_REL)
    w.close()


# the shape the paper serves (Llama-3.1-8B: hidden 4096, 32/8 heads, ffn 14336), one layer.  The weights are generated
# once per module; the oracle evaluates 3 batch rows per batch size (rows are independent in every stage), once.
_8B = {}


def _llama_8b():
    hidden, Hq, Hkv, ffn = 4096, 32, 8, 14336
    if "w" not in _8B:
        w = make_wside(hidden, Hq, Hkv, ffn, n_layers=1, max_batch=128)
        W = {which: w.weight(0, which).cpu().numpy() for which in W_STREAMS}   # device twin == gen.py: tested above
        spot = gen.gen_weight(gen.STREAM_WDOWN, 0, 2, ffn)
        assert np.array_equal(W[KF_W_DOWN][:2].view(np.uint16), spot.view(np.uint16))
        _8B.update(w=w, W=W, ref={})
    return _8B["w"], _8B["W"]


def _llama_8b_reference(batch, rows):
    w, W = _llama_8b()
    if batch not in _8B["ref"]:
        hidden, Hq = 4096, 32
        xh = gen_device.fill_x(0, batch, 0, hidden).cpu().numpy()
        o_h = gen.tensor(gen.STREAM_Q, 9, 0, np.arange(batch), Hq).transpose(1, 0, 2).astype(np.float32)
        ref = ow.project(xh[rows], W[KF_W_Q], W[KF_W_KV])
        refp = ow.post_attention(o_h.reshape(batch, -1)[rows], W[KF_W_O], W[KF_W_GATE], W[KF_W_UP], W[KF_W_DOWN])
        _8B["ref"][batch] = (o_h, ref, refp)
    return _8B["ref"][batch]


@pytest.mark.parametrize("sms", [0, 80, 64, 48, 32])
@pytest.mark.parametrize("batch", [16, 64, 128])
def test_llama_8b_layer_shape_sampled_rows(batch, sms):
    # batch x CTA count of the persistent GEMM grid = what `bench.py --pipeline` times: B_mu in {16, .., 128} with
    # kf_wside_set_sms(148 - attend_sms) in {80, 64, 48, 32}, and the default grid (0 = all SMs).  The stream-K cuts move
    # with the CTA count (e.g. 48 CTAs on gate/up: 150 k-blocks per span = the tail of a tile, a whole one, the head
    # of a third), so each combination is its own decomposition of the same contraction.
    hidden, Hq, Hkv = 4096, 32, 8
    w, _ = _llama_8b()
    rows = [0, batch // 2 - 1, batch - 1]
    o_h, ref, refp = _llama_8b_reference(batch, rows)
    w.set_sms(sms)
    x = gen_device.fill_x(0, batch, 0, hidden)
    q = torch.full((batch, Hq, 128), float("nan"), dtype=torch.float16, device="cuda")
    k = torch.full((batch, Hkv, 128), float("nan"), dtype=torch.float16, device="cuda")
    v = torch.full_like(k, float("nan"))
    w.project_q(0, x, q)
    w.project_kv(0, x, k, v)
    _close(q.cpu().numpy().reshape(batch, -1)[rows], ref["q"], f"8B q B{batch} sms{sms}")
    _close(k.cpu().numpy().reshape(batch, -1)[rows], ref["k"], f"8B k B{batch} sms{sms}")
    _close(v.cpu().numpy().reshape(batch, -1)[rows], ref["v"], f"8B v B{batch} sms{sms}")
    assert torch.isfinite(q).all() and torch.isfinite(k).all() and torch.isfinite(v).all()   # every row was written
    o = torch.from_numpy(np.ascontiguousarray(o_h)).cuda()
    xn = torch.full((batch, hidden), float("nan"), dtype=torch.float16, device="cuda")
    w.post_attention(0, o, xn)
    assert torch.isfinite(xn).all()
    _close(xn.cpu().numpy()[rows], refp["x"], f"8B x' B{batch} sms{sms}", rel=X_REL, rms_frac=X_REL)
    w.set_sms(0)


def test_llama_8b_release():
    if "w" in _8B:
        _8B["w"].close()
        _8B.clear()


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
        _close(outs[0][0][m], x.astype(np.float64), f"pipeline chain microbatch {m}", rel=CHAIN_REL, rms_frac=CHAIN_REL)
    w.close()
