"""GPU parity with POISONED KV pools: every pool byte is set to 0xFF (fp16 NaN patterns) -- and, in a second pass,
every fp16 element to 0x7C00 (+inf) -- BEFORE any request is opened or loaded.  Whatever the kernels read beyond the
valid tokens of a range (rows valid..15 of a ragged last tile, the unwritten rest of a tail range, slots never used)
is then NaN / inf, so a stale row that leaked into a score, a softmax weight or a P.V product would make an output
non-finite or push it out of tolerance.  Both kernels, fused (through the static step graph) and unfused, ragged
shapes -- last tiles with 1..15 valid rows, 1-token tail ranges, a tail range opened straight after a range fill,
every 16-token tile its own piece (min_tiles = 1) -- for 4 decode steps; every row against the fp64 oracle."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from kf_inputs.workloads import Workload  # noqa: E402
from kf_testlib import check_close, oracle_request  # noqa: E402
from paper_2606_29207_b200 import KF_IMPL_SIMPLE, KF_IMPL_TMA, KF_OK  # noqa: E402
from paper_2606_29207_b200.workload import Session  # noqa: E402

PATTERNS = {"nan_ff": 0xFFFF, "inf_7c00": 0x7C00}
STEPS = 4
# contexts at step 0 (current token included), R = 64, 16-token tiles:
#   1..15 valid rows in the last tile (1, 2, 15, 17, 31, 33, 47, 79, 191 -> 1, 2, 15, 1, 15, 1, 15, 15, 15), full tiles
#   (16, 64, 128), a 1-token tail range (65, 129), tail ranges that fill during the 4 steps (62 -> fills at step 2 and
#   opens a 1-token range at step 3; 64 -> the range is full after step 0, a new one opens at step 1; 127)
CONTEXTS = [1, 2, 15, 16, 17, 31, 33, 47, 62, 64, 65, 79, 127, 128, 129, 191]


def _poison(ses, pattern):
    for p in ses.kf.pools:
        p.view(torch.int16).fill_(pattern - 0x10000 if pattern >= 0x8000 else pattern)
    torch.cuda.synchronize()
    probe = ses.kf.pools[0][:8].view(torch.float16)
    assert not torch.isfinite(probe).any()                  # the pattern really is NaN / inf in fp16


def _check_all(wl, step, o, lse, op, lp, what):
    for r, S0 in enumerate(wl.contexts):
        S = S0 + step
        o_ref, lse_ref, op_ref, lp_ref = oracle_request(wl, 0, r, step, S, ranges=True)
        check_close(o[r], lse[r], o_ref, lse_ref, f"{what} step{step} r{r}")
        if op is not None:
            for j in range(op_ref.shape[0]):
                check_close(op[r, j], lp[r, j], op_ref[j], lp_ref[j], f"{what} step{step} r{r} range{j}")


@pytest.mark.parametrize("impl", [KF_IMPL_SIMPLE, KF_IMPL_TMA])
@pytest.mark.parametrize("pattern", list(PATTERNS), ids=list(PATTERNS))
@pytest.mark.parametrize("min_tiles", [0, 1])
def test_poisoned_pools_fused_through_the_step_graph(impl, pattern, min_tiles):
    wl = Workload("poison", 32, 8, 64, 3, CONTEXTS)
    ses = Session(wl, impl=impl, steps=STEPS, min_tiles=min_tiles)
    _poison(ses, PATTERNS[pattern])
    ses.prepare()
    kf = ses.kf
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        ins = [(ses.q_for(0, t),) + ses.kv_new_for(0, t) for t in range(STEPS)]
        g = kf.step_graph_create([0], [ins[0][0]], [ins[0][1]], [ins[0][2]], [ses.o], [ses.lse])
        for t in range(STEPS):
            ses.o.fill_(float("nan"))
            ses.lse.fill_(float("nan"))
            g.launch([ins[t][0]], [ins[t][1]], [ins[t][2]], [ses.o], [ses.lse])
            side.synchronize()
            _check_all(wl, t, ses.o.cpu().numpy(), ses.lse.cpu().numpy(), None, None, f"poison {pattern} graph")
        assert kf.status() == KF_OK
        g.destroy()
    ses.close()


@pytest.mark.parametrize("impl", [KF_IMPL_SIMPLE, KF_IMPL_TMA])
@pytest.mark.parametrize("pattern", list(PATTERNS), ids=list(PATTERNS))
@pytest.mark.parametrize("fused", [True, False, "one_launch"])
def test_poisoned_pools_eager_with_partials(impl, pattern, fused):
    wl = Workload("poison", 32, 8, 64, 3, CONTEXTS)
    ses = Session(wl, impl=impl, steps=STEPS, min_tiles=1)
    _poison(ses, PATTERNS[pattern])
    ses.prepare()
    kf = ses.kf
    for t in range(STEPS):
        kf.token_boundary()
        q = ses.q_for(0, t)
        k_new, v_new = ses.kv_new_for(0, t)
        for x in (ses.o, ses.lse, ses.o_part, ses.lse_part):
            x.fill_(float("nan"))
        ses.layer_step(0, q, k_new, v_new, fused=bool(fused), want_partials=True, one_launch=fused == "one_launch")
        kf.step_commit()
        assert kf.status() == KF_OK
        _check_all(wl, t, ses.o.cpu().numpy(), ses.lse.cpu().numpy(), ses.o_part.cpu().numpy(),
                   ses.lse_part.cpu().numpy(), f"poison {pattern} fused{fused}")
    ses.close()


def test_poisoned_pools_g8_and_long_ragged_units():
    # G = 8 (all 8 real rows of the MMA tile), ranges of 512 tokens with ragged ends, many pieces per unit
    wl = Workload("poison_g8", 64, 8, 512, 2, [1500, 700, 511, 513, 1])
    for pattern in PATTERNS.values():
        ses = Session(wl, impl=KF_IMPL_TMA, steps=2, min_tiles=1)
        _poison(ses, pattern)
        ses.prepare()
        kf = ses.kf
        for t in range(2):
            kf.token_boundary()
            q = ses.q_for(0, t)
            k_new, v_new = ses.kv_new_for(0, t)
            for x in (ses.o, ses.lse, ses.o_part, ses.lse_part):
                x.fill_(float("nan"))
            ses.layer_step(0, q, k_new, v_new, fused=True, want_partials=True, one_launch=t == 1)
            kf.step_commit()
            assert kf.status() == KF_OK
            _check_all(wl, t, ses.o.cpu().numpy(), ses.lse.cpu().numpy(), ses.o_part.cpu().numpy(),
                       ses.lse_part.cpu().numpy(), "poison_g8")
        ses.close()
